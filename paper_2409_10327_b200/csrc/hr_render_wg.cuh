// hr_render_wg.cuh -- the fused render_frame kernel (steps a1-a11) on tcgen05 / TMEM, warpgroup-multiplexed.
//
// One persistent CTA per SM holds G independent 128-thread warpgroups (WG).  A WG is the 128 TMEM lanes of its own
// TMEM column range: thread r owns row r of every 128 x N tcgen05.mma the WG issues, so an MLP activation never
// crosses threads.  The G warpgroups share the UMMA weight tiles in shared memory, are scheduled independently
// (named barriers + one mbarrier each) and hide each other's MMA / gather / barrier latencies: with G = 4 every SM
// sub-partition has four warps to pick from instead of two.
//
// Per 128-pixel tile a WG runs
//   A   primary point: f = H(x) (fp32, hi/lo split), P = W1f f + b1, n,a,r = B(f)                     (a1-a5)
//   A2  direct set: v = I(f, w_s) per direction, Eq. 1 with the env map                                (a6, a9-a11)
//   B   secondary set: (v, t) = I(f, w_j) in split precision, x' = x + t w_j, and the weight
//       g_j = (1 - v_j) f_r (n.w_j)^+ / (p_j S_i S_2) of L'_o in Eq. 2.  Every ray with a non-zero weight
//       becomes a 48-byte work item in the WG's ring (only occluded rays are traced further;
//       HR_DENSE keeps every ray)                                                                      (a6, a7)
//   C   items are drained 128 at a time, one per thread, whoever produced them: f' = H(x'), P' = W1f f' + b1,
//       n',a',r' = B(f'), v'_k = I(f', w'_k) over the tertiary set, L'_o (Eq. 1 with w_o' = -w_j); the weighted
//       radiance is added to the owner pixel's accumulator in shared memory                           (a8)
//   D   rgb = direct + indirect                                                                        (a11)
//
// PREC = 0: fp16 activations (BASELINE.json configs[3]); the primary point and the secondary trace, whose t moves
//           x', run in split precision (hi + lo fp16, SURVEY 8(c) conditioning note).
// PREC = 1: fp32-grade arithmetic on the fp16 tensor cores for mlp_dtype == HR_F32: every activation AND every
//           weight is split x = hi + lo (both fp16), each layer is three MMA passes hi*Whi + lo*Whi + hi*Wlo with
//           fp32 accumulation (the dropped lo*lo term is 2^-22 relative), epilogues and shading in fp32.
#pragma once
#include <cstring>

#include "hr_kernels_ffma.cuh"
#include "hr_kernels_tc.cuh"

namespace hr {
namespace wg {
using namespace hr::tc;

constexpr int kRows = 128;                    // rows (threads) per warpgroup
constexpr int kRing = 2048;                   // work items per WG ring (power of two, >= 127 + kChunkJ * 128)
constexpr int kChunkJ = 8;                    // secondary directions traced between two drains
constexpr int kMaxG = 4;
constexpr int kMaxS2 = tc::kMaxS2;              // shared tertiary set staged in shared memory
constexpr int kHiTileBytes = kNumTiles * kTileBytes + kTile3Bytes;       // 34 KB: I.W1f, B.W1, I.W2, B.W2, B.W3

struct __align__(16) Item {                   // one secondary hit waiting for its L'_o
  float x, y, z, wx;                          // x' and the direction it was reached along (w_o' = -w)
  float wy, wz, gr, gg;                       // weight of L'_o in the owner's pixel, per channel
  float gb; uint32_t owner; uint32_t pad0, pad1;   // owner = row | j << 8
};
static_assert(sizeof(Item) == 48, "Item is three 16-byte words");

template <int PREC, int G> struct Cols {
  static_assert(G >= 1 && G <= kMaxG, "1..4 warpgroups");
  static constexpr uint32_t stride = G == 4 ? 128u : (G == 3 ? 168u : (G == 2 ? 256u : 512u));
  // A = columns 0..63 (fp16 pairs): 0..31 for the fp16 layers, hi | lo for the split layers.  D = 64 fp32 accumulator columns.
  // The constant operand of the bias K-steps, rows of [1, 1, 0 .. 0], lives in SHARED memory (kOnesBytes of identical
  // 16-byte chunks, so the swizzle cannot matter), which leaves all 128 columns of a G = 4 warpgroup to A and D.
  static constexpr uint32_t d = 64u;
};
constexpr int kOnesBytes = 128 * 128;         // a 128-row K-major SWIZZLE_128B tile of uniform chunks

struct WgCtx {
  uint32_t tmem;      // TMEM address of the WG's column 0, lane 0
  uint32_t lane;      // this warp's lane base << 16
  uint32_t mbar;      // shared address of the WG's mbarrier
  uint32_t phase;
  uint32_t tile0;     // shared address of the weight tiles
  uint32_t lo_off;    // byte offset of the lo tiles (PREC = 1)
  uint32_t ones;      // shared address of the uniform bias operand
  int bar_id;         // named barrier of the WG
  int t;              // thread index in the WG
  mutable uint32_t rot;   // layers issued so far
  uint32_t rot_mask;      // 3: the issuing warp rotates over the four warps of the group (k_render_wg); 0: always warp 0 (k_trace_wg)
};

__device__ __forceinline__ void tmem_st4(uint32_t taddr, const uint32_t (&r)[4]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
}
__device__ __forceinline__ void tmem_stN(uint32_t taddr, const uint32_t (&r)[4]) { tmem_st4(taddr, r); }
__device__ __forceinline__ void tmem_stN(uint32_t taddr, const uint32_t (&r)[2]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(taddr), "r"(r[0]), "r"(r[1]) : "memory");
}
__device__ __forceinline__ void tmem_stN(uint32_t taddr, const uint32_t (&r)[1]) { tmem_st1(taddr, r[0]); }
__device__ __forceinline__ void wg_sync(const WgCtx& c) { asm volatile("bar.sync %0, 128;" ::"r"(c.bar_id) : "memory"); }

// One 128 x N layer of the WG: D = A W^T (+ bias K-step).  A = `ksteps` K-steps of fp16 at column a_col; split_a: a lo
// block follows the hi block; PREC = 1 adds the pass against the lo weights.  All threads must have stored their A rows.
template <int PREC, int G>
__device__ __forceinline__ void issue_layer(const WgCtx& c, uint32_t a_col, int tile, int ksteps, bool split_a, int bias_tile,
                                            int bias_kstep, uint32_t idesc = kIdesc, uint32_t d_col = Cols<PREC, G>::d) {
  wait_st();
  fence_before();
  // The issuing warp rotates from layer to layer: warp w of every group sits on SM sub-partition w, so a fixed issuer would put
  // the barrier wait and the MMA issue of all G groups on one scheduler (C2 dense 23.1 -> 22.9 ms, compacted 10.9 -> 10.65,
  // C3 compacted 7.54 -> 7.38; k_trace_wg measured slower with it, 5.77 -> 6.24 ms, and keeps warp 0).
  const uint32_t iw = (c.rot++) & c.rot_mask;
  if ((uint32_t)(c.t >> 5) != iw) {             // three warps only announce their rows and go on to the work that needs no D
    asm volatile("bar.arrive %0, 128;" ::"r"(c.bar_id) : "memory");
  } else {                                      // the issuing warp, converged; one elected lane issues
    wg_sync(c);
    fence_after();
    const uint32_t d = c.tmem + d_col;
    const uint32_t a = c.tmem + a_col;
    const uint64_t bd = make_bdesc(c.tile0 + tile * kTileBytes);
    for (int k = 0; k < ksteps; ++k) mma_f16_ts_elect(d, a + 8 * k, bd + 2 * k, idesc, k > 0);
    if (split_a)
      for (int k = 0; k < ksteps; ++k) mma_f16_ts_elect(d, a + 8 * (ksteps + k), bd + 2 * k, idesc, 1u);
    if (PREC == 1) {
      const uint64_t bl = make_bdesc(c.tile0 + c.lo_off + tile * kTileBytes);
      for (int k = 0; k < ksteps; ++k) mma_f16_ts_elect(d, a + 8 * k, bl + 2 * k, idesc, 1u);
    }
    if (bias_tile >= 0)          // D += [1,1,0..|1,1,0..] x K-step: columns 0,1 hold the bias hi/lo, columns 8,9 are zero
      mma_f16_ss_elect(d, make_bdesc(c.ones), make_bdesc(c.tile0 + bias_tile * kTileBytes) + 2 * bias_kstep, idesc, 1u);
    mma_commit_elect(c.mbar);
  }
}
// every 16-byte chunk of the bias operand = fp16 [1, 1, 0, 0, 0, 0, 0, 0]
__device__ __forceinline__ void fill_ones(uint8_t* s_ones, int nthreads) {
  uint4* dst = reinterpret_cast<uint4*>(s_ones);
  for (int i = threadIdx.x; i < kOnesBytes / 16; i += nthreads) dst[i] = make_uint4(0x3C003C00u, 0u, 0u, 0u);
}
__device__ __forceinline__ void wait_layer(WgCtx& c) {
  mbar_wait(c.mbar, c.phase);
  c.phase ^= 1u;
  fence_after();
}

// ---------------------------------------------------------------------------------------------------- row stages
// packed fp32 pairs (sm_100 FFMA2 / FADD2): one issue slot for two lanes of fp32 work.  A scalar multiplicand is passed
// twice and ptxas folds it into the broadcast form of the instruction; constant-bank pairs ride as uniform-register operands.
__device__ __forceinline__ void fma2(float a0, float a1, float b0, float b1, float& c0, float& c1) {
  asm("{\n\t.reg .b64 a, b, c;\n\tmov.b64 a, {%2, %3};\n\tmov.b64 b, {%4, %5};\n\tmov.b64 c, {%0, %1};\n\t"
      "fma.rn.f32x2 c, a, b, c;\n\tmov.b64 {%0, %1}, c;\n\t}"
      : "+f"(c0), "+f"(c1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}
__device__ __forceinline__ void add2(float a0, float a1, float b0, float b1, float& c0, float& c1) {
  asm("{\n\t.reg .b64 a, b, c;\n\tmov.b64 a, {%2, %3};\n\tmov.b64 b, {%4, %5};\n\tadd.rn.f32x2 c, a, b;\n\tmov.b64 {%0, %1}, c;\n\t}"
      : "=f"(c0), "=f"(c1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}
__device__ __forceinline__ void sub2(float a0, float a1, float b0, float b1, float& c0, float& c1) {
  asm("{\n\t.reg .b64 a, b, c;\n\tmov.b64 a, {%2, %3};\n\tmov.b64 b, {%4, %5};\n\tsub.rn.f32x2 c, a, b;\n\tmov.b64 {%0, %1}, c;\n\t}"
      : "=f"(c0), "=f"(c1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}
// fp32 pair -> hi fp16x2 word and the fp16x2 word of the residual.  hi is the fp32 value with its low 13 mantissa bits cleared
// (10 kept = fp16's, so the conversion is exact inside the fp16 normal range the split_ok check of hashrender_create
// guarantees), the residual a - hi is exact in fp32 and is rounded once to fp16: a = hi + lo to 2^-21 relative.
__device__ __forceinline__ void split_pair(float a0, float a1, uint32_t& hi, uint32_t& lo) {
  const float m0 = __uint_as_float(__float_as_uint(a0) & 0xFFFFE000u), m1 = __uint_as_float(__float_as_uint(a1) & 0xFFFFE000u);
  float l0, l1;
  sub2(a0, a1, m0, m1, l0, l1);
  hi = pack_rn(m0, m1);
  lo = pack_rn(l0, l1);
}
// the same split of (max(a0, 0), max(a1, 0)): truncation keeps the sign of a and of a - hi, so the relu rides in both conversions
__device__ __forceinline__ void split_pair_relu(float a0, float a1, uint32_t& hi, uint32_t& lo) {
  const float m0 = __uint_as_float(__float_as_uint(a0) & 0xFFFFE000u), m1 = __uint_as_float(__float_as_uint(a1) & 0xFFFFE000u);
  float l0, l1;
  sub2(a0, a1, m0, m1, l0, l1);
  hi = pack_relu(m0, m1);
  lo = pack_relu(l0, l1);
}

// z_v = b3 + w3v . relu(D) with fp16x2 FMAs (b2 rode in the MMA); PREC = 0 direct / tertiary queries
__device__ __forceinline__ float epi_fast(uint32_t tD, const TcConst& cw) {
  __half2 acc[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) acc[q] = __float2half2_rn(0.f);
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
  const float2 f = __half22float2(__hadd2(__hadd2(acc[0], acc[1]), __hadd2(acc[2], acc[3])));
  return cw.b3[0] + (f.x + f.y);
}
// fp32 epilogues (b2 rode in the MMA as a hi/lo bias K-step unless ADD_B2)
template <bool ADD_B2>
__device__ __forceinline__ void epi_precise(uint32_t tD, const TcConst& cw, float& zv, float& zt) {
  float z0[4] = {cw.b3[0], 0.f, 0.f, 0.f}, z1[4] = {cw.b3[1], 0.f, 0.f, 0.f};
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 32; k += 2) {
      const float a0 = fmaxf(ADD_B2 ? __uint_as_float(r[k]) + cw.b2[32 * h + k] : __uint_as_float(r[k]), 0.f);
      const float a1 = fmaxf(ADD_B2 ? __uint_as_float(r[k + 1]) + cw.b2[32 * h + k + 1] : __uint_as_float(r[k + 1]), 0.f);
      fma2(cw.w3[0][32 * h + k], cw.w3[0][32 * h + k + 1], a0, a1, z0[k & 2], z0[(k & 2) + 1]);
      fma2(cw.w3[1][32 * h + k], cw.w3[1][32 * h + k + 1], a0, a1, z1[k & 2], z1[(k & 2) + 1]);
    }
  }
  zv = (z0[0] + z0[1]) + (z0[2] + z0[3]);
  zt = (z1[0] + z1[1]) + (z1[2] + z1[3]);
}
__device__ __forceinline__ float epi_precise_v(uint32_t tD, const TcConst& cw) {
  float z0[4] = {cw.b3[0], 0.f, 0.f, 0.f};
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 32; k += 2)
      fma2(cw.w3[0][32 * h + k], cw.w3[0][32 * h + k + 1], fmaxf(__uint_as_float(r[k]), 0.f), fmaxf(__uint_as_float(r[k + 1]), 0.f),
           z0[k & 2], z0[(k & 2) + 1]);
  }
  return (z0[0] + z0[1]) + (z0[2] + z0[3]);
}

// relu(D) -> A columns 0..31 (fp16) or 0..31 | 32..63 (hi | lo)
template <bool SPLIT>
__device__ __forceinline__ void hidden_to_A(uint32_t tD, uint32_t tA) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
    uint32_t p[16], q[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      if (SPLIT) split_pair_relu(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]), p[k], q[k]);
      else p[k] = pack_relu(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
    }
    tmem_st16(tA + 16 * h, p);
    if (SPLIT) tmem_st16(tA + 32 + 16 * h, q);
  }
}

// h1 = relu(P + W1w . w) -> A; P4(q) yields the layer-1 partials of hidden units 4q .. 4q+3 (one LDS.128)
template <bool SPLIT, typename PF>
__device__ __forceinline__ void h1_dir(uint32_t tA, const TcConst& cw, PF P4, float wx, float wy, float wz) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t p[16], q[16];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float4 pv = P4(8 * h + k);
      const float pin[4] = {pv.x, pv.y, pv.z, pv.w};
      float a[4] = {pin[0], pin[1], pin[2], pin[3]};
#pragma unroll
      for (int e = 0; e < 4; e += 2) {
        const int j = 32 * h + 4 * k + e;
        fma2(cw.w1w[0][j], cw.w1w[0][j + 1], wx, wx, a[e], a[e + 1]);
        fma2(cw.w1w[1][j], cw.w1w[1][j + 1], wy, wy, a[e], a[e + 1]);
        fma2(cw.w1w[2][j], cw.w1w[2][j + 1], wz, wz, a[e], a[e + 1]);
      }
      if (SPLIT) {
        split_pair_relu(a[0], a[1], p[2 * k], q[2 * k]);
        split_pair_relu(a[2], a[3], p[2 * k + 1], q[2 * k + 1]);
      } else {
        p[2 * k] = pack_relu(a[0], a[1]);
        p[2 * k + 1] = pack_relu(a[2], a[3]);
      }
    }
    tmem_st16(tA + 16 * h, p);
    if (SPLIT) tmem_st16(tA + 32 + 16 * h, q);
  }
}
// D (64 fp32 columns) -> this thread's column of a [16][128] float4 array in shared memory
__device__ __forceinline__ void store_D_f4(uint32_t tD, float4* dst) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 8; ++k)
      dst[(8 * h + k) * kRows] = make_float4(__uint_as_float(r[4 * k]), __uint_as_float(r[4 * k + 1]), __uint_as_float(r[4 * k + 2]),
                                             __uint_as_float(r[4 * k + 3]));
  }
}
// shared tertiary set, PREC = 0: P and Q = W1w . w'_k both fp16 pairs, one fma.relu per pair
__device__ __forceinline__ void h1_shared_h2(uint32_t tA, const uint32_t (&Ph)[kH / 2], const uint32_t* __restrict__ Qh) {
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
// shared tertiary set, PREC = 1: fp32 P (registers) + fp32 Q (shared memory), split
__device__ __forceinline__ void h1_shared_split(uint32_t tA, const float (&P)[kH], const float* __restrict__ Q) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t p[16], q[16];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float4 v = reinterpret_cast<const float4*>(Q)[8 * h + k];
      const int j = 32 * h + 4 * k;
      float a[4];
      add2(P[j], P[j + 1], v.x, v.y, a[0], a[1]);
      add2(P[j + 2], P[j + 3], v.z, v.w, a[2], a[3]);
      split_pair_relu(a[0], a[1], p[2 * k], q[2 * k]);
      split_pair_relu(a[2], a[3], p[2 * k + 1], q[2 * k + 1]);
    }
    tmem_st16(tA + 16 * h, p);
    tmem_st16(tA + 32 + 16 * h, q);
  }
}

template <int N>
__device__ __forceinline__ void load_D_f32(uint32_t tD, float (&P)[N]) {
  static_assert(N == kH, "64 accumulator columns");
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 32; ++k) P[32 * h + k] = __uint_as_float(r[k]);
  }
}
__device__ __forceinline__ void load_D_h2(uint32_t tD, uint32_t (&Ph)[kH / 2]) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 16; ++k) Ph[16 * h + k] = pack_rn(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
  }
}

// One level of the fp32 encode in two halves, so that the caller can put a whole tertiary query between the gathers and
// their first use (the arithmetic is encode_level's).
template <bool F16TAB> struct Taps32;
template <> struct Taps32<false> { float2 v[8]; float w[3]; __device__ __forceinline__ float2 tap(int k) const { return v[k]; } };
template <> struct Taps32<true> {                          // fp16 rows stay packed (one register each) until they are interpolated
  uint32_t r[8]; float w[3];
  __device__ __forceinline__ float2 tap(int k) const { return __half22float2(*reinterpret_cast<const __half2*>(&r[k])); }
};
template <bool F16TAB>
__device__ __forceinline__ void gather32(const GridP& g, int l, float x, float y, float z, Taps32<F16TAB>& t) {
  const uint32_t N = g.res[l];
  const Cell c = cell_of(N, x, y, z);
  if constexpr (F16TAB) gather8_h2(g, l, c.c0, t.r); else gather8_f2(g, l, c.c0, t.v);
  t.w[0] = c.w[0]; t.w[1] = c.w[1]; t.w[2] = c.w[2];
}
// trilinear interpolation of the taps: the arithmetic (and its order) is encode_level's
template <bool F16TAB>
__device__ __forceinline__ float2 lerp32(const Taps32<F16TAB>& t) {
  const float wx[2] = {1.f - t.w[0], t.w[0]}, wy[2] = {1.f - t.w[1], t.w[1]}, wz[2] = {1.f - t.w[2], t.w[2]};
  float2 f = make_float2(0.f, 0.f);
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const float wt = wx[k & 1] * wy[(k >> 1) & 1] * wz[(k >> 2) & 1];
    const float2 v = t.tap(k);
    f.x = fmaf(wt, v.x, f.x);
    f.y = fmaf(wt, v.y, f.y);
  }
  return f;
}
// f = H(x) in fp32 -> A columns 0..15 (hi) | 16..31 (lo), LIF levels per TMEM store
template <bool F16TAB, int LIF, int PAIR = -1>
__device__ __forceinline__ void encode_split_to(uint32_t tA, const GridP& g, float x, float y, float z, float* scr = nullptr,
                                                const L2Pol* pol = nullptr) {
#pragma unroll 1
  for (int l0 = 0; l0 < kMaxL; l0 += LIF) {
    uint32_t hi[LIF], lo[LIF];
#pragma unroll
    for (int q = 0; q < LIF; ++q) {
      // The branch is kept although null levels (GridP) would read zeros without it: it keeps each level's eight gathers
      // and their interpolation in a block of their own.  Without it the compiler hoists all 8 LIF gathers of the group above the
      // first use, and that burst is SLOWER (k_trace_wg, C4 at 2^24 points: T = 2^19 5.8 -> 7.5 ms, T = 2^24 13.5 -> 16.1 ms;
      // written out as explicit gather / interpolate phases: 7.7 / 16.8 ms) -- L1 serves a warp's 32 divergent lines one per
      // cycle, and 16 warps x 32 loads queue behind each other instead of overlapping with the interpolation of the others.
      hi[q] = 0u; lo[q] = 0u;
      if (l0 + q < (int)g.L) {
        const float2 v = encode_level<F16TAB, PAIR>(g, l0 + q, x, y, z, nullptr, nullptr, pol);
        split_pair(v.x, v.y, hi[q], lo[q]);
        if (scr) { scr[(2 * (l0 + q)) * kRows] = v.x; scr[(2 * (l0 + q) + 1) * kRows] = v.y; }
      } else if (scr) {
        scr[(2 * (l0 + q)) * kRows] = 0.f; scr[(2 * (l0 + q) + 1) * kRows] = 0.f;
      }
    }
    tmem_stN(tA + l0, hi);
    tmem_stN(tA + 16 + l0, lo);
  }
}
// fast encode of a secondary point (already clamped) -> A columns 0..15, fp16 pairs
template <bool F16TAB, int LIF>
__device__ __forceinline__ void encode_fast_to(uint32_t tA, const GridP& g, float x, float y, float z) {
#pragma unroll 1
  for (int l0 = 0; l0 < kMaxL; l0 += LIF) {               // LIF levels (8 LIF gathers) in flight
    LevelTaps<F16TAB> t[LIF];
#pragma unroll
    for (int q = 0; q < LIF; ++q) gather_level<F16TAB>(g, l0 + q, x, y, z, t[q]);
    uint32_t f[LIF];
#pragma unroll
    for (int q = 0; q < LIF; ++q) f[q] = lerp_level(t[q]);
    tmem_stN(tA + l0, f);
  }
}

// interpolate, split, store the level's fp16x2 words to TMEM columns tF + l (hi) and tF + 16 + l (lo)
template <bool F16TAB>
__device__ __forceinline__ void finish32(uint32_t tF, int l, const Taps32<F16TAB>& t) {
  const float2 f = lerp32(t);
  uint32_t hi, lo;
  split_pair(f.x, f.y, hi, lo);
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(tF + l), "r"(hi) : "memory");
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(tF + 16 + l), "r"(lo) : "memory");
}

// B over the features at A columns 0.. (hi | lo when PREC = 1): all three layers on the tensor core, biases of layers 1-2
// ride as K-steps, layer 3 is an N = 16 MMA over the zero-padded 7-row W3; b3 is added in registers.
template <int PREC, int G>
__device__ __forceinline__ void brdf_mma(WgCtx& c, const TcConst& cw, const ShadeP& sp, float (&b)[7], uint32_t f_col = 0,
                                         bool l1_done = false) {
  const uint32_t tA = c.tmem + c.lane, tD = c.tmem + c.lane + Cols<PREC, G>::d;
  if (!l1_done) {                               // l1_done: the caller's N = 128 MMA has already left layer 1 in D
    issue_layer<PREC, G>(c, f_col, 1, 2, PREC == 1, 1, 2);
    wait_layer(c);
  }
  hidden_to_A<PREC == 1>(tD, tA);
  issue_layer<PREC, G>(c, 0, 3, 4, PREC == 1, 1, 3);
  wait_layer(c);
  hidden_to_A<PREC == 1>(tD, tA);
  issue_layer<PREC, G>(c, 0, 4, 4, PREC == 1, -1, 0, kIdescN16);
  wait_layer(c);
  uint32_t r[8];
  tmem_ld8(tD, r);
  wait_ld();
  float o[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) o[q] = __uint_as_float(r[q]) + cw.Bb3[q];
  brdf_maps(sp, o, b);
}

// Primary point (once per pixel): B in split precision with layer 3 in fp32 registers (n = o/||o|| amplifies an absolute
// error of o and every sample of the pixel sees the same n).  f (hi | lo) must sit in A columns 0..31.
template <int PREC, int G>
__device__ __forceinline__ void brdf_primary(WgCtx& c, const TcConst& cw, const ShadeP& sp, float (&b)[7]) {
  const uint32_t tA = c.tmem + c.lane, tD = c.tmem + c.lane + Cols<PREC, G>::d;
  issue_layer<PREC, G>(c, 0, 1, 2, true, 1, 2);
  wait_layer(c);
  hidden_to_A<true>(tD, tA);
  issue_layer<PREC, G>(c, 0, 3, 4, true, 1, 3);
  wait_layer(c);
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

// ---------------------------------------------------------------------------------------------------- shared memory
template <int PREC, bool TSHARED, int G> struct SmemPlan {
  static constexpr bool p2_in_smem = !TSHARED;                       // per-point tertiary sets keep P' in shared memory
  static constexpr size_t tiles = (size_t)kHiTileBytes * (PREC ? 2 : 1);
  static constexpr size_t per_wg = (size_t)kH * kRows * 4 * (p2_in_smem ? 2 : 1)      // Ps (+ P2s)
                                   + kRows * 4 * 4                                     // acc[128][4]
                                   + 64;                                               // queue head/tail, tile slot
  static constexpr size_t shared_set = (size_t)kMaxS2 * kH * 4 + kMaxS2 * 8 * 4;      // Qt, Lt
  static constexpr size_t bytes = 1024 + tiles + kOnesBytes + G * per_wg + shared_set + 8 * kMaxG + 16;
};

// ---------------------------------------------------------------------------------------------------- the kernel
// counters[0]: next tile (zeroed before every launch); [1]: items evaluated; [2]: secondary rays traced (dense count)
// IND = false: frames without the indirect term (BASELINE configs[1]): phases B and C are compiled out, which takes the
// split-precision kernel from 168 to <= 128 registers and lets four warpgroups share an SM instead of three.
template <bool F16TAB, int PREC, bool TSHARED, int G, bool IND = true>
__global__ void __launch_bounds__(kRows* G, 1)
    k_render_wg(const __grid_constant__ GridP g, EnvP env, ShadeP sp, const __grid_constant__ TcConst cw, const uint8_t* __restrict__ wtiles,
                const float* __restrict__ wts32, FrameP fr, float* __restrict__ rgb, Item* __restrict__ ring,
                unsigned long long* __restrict__ counters) {
  using CL = Cols<PREC, G>;
#ifdef HR_LIF
  constexpr int LIF = HR_LIF;
#else
  // levels whose gathers are issued together in the encodes of this kernel.  Two since the coarsest levels are cell-major (one
  // load each): same box, C3 dense 15.22 -> 15.00 ms, C2 dense 23.13 -> 23.07, compacted frames and C1 unchanged.  Before the
  // cell-major levels one level at a time was best (C3 dense / compacted, C2 compacted, ms: LIF 1 15.65 / 7.61 / 10.87, LIF 2
  // (G = 4) and 4 (G = 3) 16.12 / 7.72 / 11.36, LIF 4 at G = 4 19.99 / 9.62): the L1 passes one missing sector per cycle to the L2,
  // so a burst of gathers from every warp queues up instead of overlapping with the other warps' arithmetic.
  constexpr int LIF = 2;
#endif
  using SP = SmemPlan<PREC, TSHARED, G>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* sp0 = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint8_t* s_tiles = sp0;
  uint8_t* s_ones = s_tiles + SP::tiles;
  uint8_t* s_wg = s_ones + kOnesBytes;
  float* s_Qt = reinterpret_cast<float*>(s_wg + G * SP::per_wg);
  float* s_Lt = s_Qt + kMaxS2 * kH;
  uint64_t* s_mbar = reinterpret_cast<uint64_t*>(s_Lt + kMaxS2 * 8);
  uint32_t* s_tmem = reinterpret_cast<uint32_t*>(s_mbar + kMaxG);

  const int wgi = threadIdx.x / kRows;
  const int warp = threadIdx.x >> 5;
  WgCtx c;
  c.t = threadIdx.x % kRows;
  c.bar_id = 1 + wgi;
  c.rot = 0; c.rot_mask = 3u;
  // ---- setup: TMEM (the CTA owns all 512 columns), mbarriers, weight tiles -----------------------------------------
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (threadIdx.x < G) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(s_mbar + threadIdx.x)) : "memory");
  if (threadIdx.x == 0) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  {
    const uint4* src = reinterpret_cast<const uint4*>(wtiles);
    uint4* dst = reinterpret_cast<uint4*>(s_tiles);
    for (int i = threadIdx.x; i < (int)(SP::tiles / 16); i += kRows * G) dst[i] = __ldg(src + i);
  }
  fill_ones(s_ones, kRows * G);
  const bool indirect = IND && (fr.flags & 4u) && fr.s.S && fr.t.S;
  if (indirect && TSHARED) {                    // shared tertiary set: Q_k = W1w . w'_k; per k: radiance, pdf, direction
    for (int e = threadIdx.x; e < (int)fr.t.S * kH; e += kRows * G) {
      const int k = e / kH, q = e % kH;
      const float* dp = fr.t.dir + 3 * k;
      const float qv = cw.w1w[0][q] * __ldg(dp) + cw.w1w[1][q] * __ldg(dp + 1) + cw.w1w[2][q] * __ldg(dp + 2);
      if (PREC == 0) reinterpret_cast<__half*>(s_Qt)[e] = __float2half_rn(qv);
      else s_Qt[e] = qv;
    }
    for (int k = threadIdx.x; k < (int)fr.t.S; k += kRows * G) {
      const float* dp = fr.t.dir + 3 * k;
      const float tx = __ldg(dp), ty = __ldg(dp + 1), tz = __ldg(dp + 2);
      float3 L;
      if (fr.t.Lin) L = make_float3(__ldg(fr.t.Lin + 3 * k), __ldg(fr.t.Lin + 3 * k + 1), __ldg(fr.t.Lin + 3 * k + 2));
      else L = env_lookup(env, tx, ty, tz);
      float* o = s_Lt + 8 * k;
      o[0] = L.x; o[1] = L.y; o[2] = L.z; o[3] = __ldg(fr.t.pdf + k); o[4] = tx; o[5] = ty; o[6] = tz; o[7] = 0.f;
    }
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy tile writes -> visible to the tensor core
  fence_before();
  __syncthreads();
  fence_after();
  // warp-uniform by construction; the reductions tell the compiler so, which keeps the MMA operands (TMEM addresses, smem
  // descriptors, the mbarrier) in uniform registers instead of re-broadcasting them from a lane before every tcgen05.mma
  c.tmem = __reduce_min_sync(0xFFFFFFFFu, *s_tmem + CL::stride * wgi);
  c.lane = __reduce_min_sync(0xFFFFFFFFu, (uint32_t)((warp & 3) * 32) << 16);     // tcgen05.ld / st addresses are uniform operands too
  c.mbar = __reduce_min_sync(0xFFFFFFFFu, smem_u32(s_mbar + wgi));
  c.phase = 0;
  c.tile0 = __reduce_min_sync(0xFFFFFFFFu, smem_u32(s_tiles));
  c.lo_off = kHiTileBytes;
  c.ones = __reduce_min_sync(0xFFFFFFFFu, smem_u32(s_ones));
  const uint32_t tA = c.tmem + c.lane, tD = c.tmem + c.lane + CL::d;
  uint8_t* my = s_wg + wgi * SP::per_wg;
  float* Ps = reinterpret_cast<float*>(my) + c.t;                                     // Ps[k * 128]
  float4* Ps4 = reinterpret_cast<float4*>(my) + c.t;                                  // the same memory as [16][128] float4
  float4* P2s4 = SP::p2_in_smem ? Ps4 + (kH / 4) * kRows : nullptr;
  float* acc = reinterpret_cast<float*>(my + (size_t)kH * kRows * 4 * (SP::p2_in_smem ? 2 : 1));
  uint32_t* qctl = reinterpret_cast<uint32_t*>(acc + kRows * 4);                      // [0] head, [1] tail, [2] tile
  Item* myring = ring + ((size_t)blockIdx.x * G + wgi) * kRing;
  if (c.t == 0) { qctl[0] = 0u; qctl[1] = 0u; }
  const unsigned long long ntiles = (fr.N + kRows - 1) / kRows;
  const int S_i = indirect ? (int)fr.s.S : 0;
  const uint32_t S2 = fr.t.S;
  const bool dense = fr.flags & 8u;
  const bool shadow = fr.flags & 2u;
  uint32_t n_items = 0, n_rays = 0;
  uint32_t head = 0;                                                                  // mirrored in registers (uniform in the WG)

  // ---- phase C: one 128-item group, one item per thread -------------------------------------------------------------
  // Split-precision kernel at G = 3: the warpgroup's 168 TMEM columns leave 40 beside A and D.  Columns 128..159 hold the
  // features f' (hi | lo) of a group, and while a group runs its tertiary queries it encodes the NEXT group's points into
  // them, two levels per query: the gathers of a level are issued before the query's row arithmetic / MMA wait and used
  // after it, so their L2 latency costs nothing (it was 19 % of the kernel's stall samples).
  // (The fp16 kernel has columns 32..63 free and the code below serves it too, but at its 128-register budget the extra
  // live taps spill and its queries are too short to cover a gather: measured 18.5 ms against 16.7 ms, so it stays off.)
  constexpr bool kPre = TSHARED && PREC == 1 && G == 3;
  constexpr uint32_t kFCol = !kPre ? 0u : (PREC == 1 ? 128u : 32u);
  const uint32_t tF = tA + kFCol;
  bool pre_done = false;                                                              // tF holds the features of the next group
  auto drain_group = [&](uint32_t count, unsigned long long tile_base, uint32_t next_count) {
    const bool on = (uint32_t)c.t < count;
    float ix = 0.5f, iy = 0.5f, iz = 0.5f, iwx = 0.f, iwy = 0.f, iwz = 1.f, wr = 0.f, wgc = 0.f, wb = 0.f;
    uint32_t owner = 0;
    if (on) {
      const float4* ip = reinterpret_cast<const float4*>(myring + ((head + c.t) & (kRing - 1)));
      const float4 a = __ldcg(ip), b4 = __ldcg(ip + 1), c4 = __ldcg(ip + 2);
      ix = a.x; iy = a.y; iz = a.z; iwx = a.w; iwy = b4.x; iwz = b4.y; wr = b4.z; wgc = b4.w; wb = c4.x;
      owner = __float_as_uint(c4.y);
    }
    // a1-a4 at x', then P' = W1f f' + b1
    if (PREC == 1) { if (!(kPre && pre_done)) encode_split_to<F16TAB, LIF>(tF, g, ix, iy, iz); }
    else { if (!(kPre && pre_done)) encode_fast_to<F16TAB, LIF>(tF, g, ix, iy, iz); }
    // kPre: the features sit outside columns 0..127, so P' (I.W1f, tile 0) and layer 1 of B (B.W1, tile 1: the next 64 rows of
    // the same shared-memory tile, its bias in the same K-step) are ONE N = 128 MMA set into columns 0..127: P' lands in
    // 0..63, B's layer 1 in 64..127 where D always is -- one barrier / commit / wait round trip less per group.
    if constexpr (kPre) issue_layer<PREC, G>(c, kFCol, 0, 2, true, 0, 2, kIdescN128, 0u);
    else issue_layer<PREC, G>(c, kFCol, 0, 2, PREC == 1, 0, 2);
    // the next group's points (kPre): positions only, the rest of the item is read when its turn comes
    float nx = 0.5f, ny = 0.5f, nz = 0.5f;
    const bool pre = kPre && next_count > 0u && S2 >= 8u;                              // WG-uniform
    if (pre && (uint32_t)c.t < next_count) {
      const float4 a = __ldcg(reinterpret_cast<const float4*>(myring + ((head + count + c.t) & (kRing - 1))));
      nx = a.x; ny = a.y; nz = a.z;
    }
    wait_layer(c);
    uint32_t P2h[kH / 2];                                             // only the one the instantiation uses survives
    float P2[kH];
    if constexpr (TSHARED) {
      if constexpr (PREC == 0) load_D_h2(tD, P2h); else load_D_f32(kPre ? tA : tD, P2);
    } else {
      store_D_f4(tD, P2s4);
    }
    float bb[7];
    brdf_mma<PREC, G>(c, cw, sp, bb, kFCol, kPre);                    // a5 at x' (the feature columns still hold f')
    // a8: Eq. 1 at x' over the tertiary set, w_o' = -w_j
    const unsigned long long trow = TSHARED ? 0ull : (tile_base + (owner & 0xFFu)) * (unsigned long long)fr.s.S + (owner >> 8);
    float lr = 0.f, lg = 0.f, lb = 0.f;
    for (uint32_t k = 0; k < S2; ++k) {
      float tx, ty, tz, tpdf;
      float3 L;
      Taps32<F16TAB> taps;                                            // PREC 1: fp32 taps; PREC 0: fp16x2 taps (only one survives)
      LevelTaps<F16TAB> htaps;
      // levels l >= g.L are null levels of the device layout (zero rows, GridP): they gather zeros, never past the allocation
      auto pre_gather = [&](int l) {
        if constexpr (PREC == 1) gather32<F16TAB>(g, l, nx, ny, nz, taps); else gather_level<F16TAB>(g, l, nx, ny, nz, htaps);
      };
      auto pre_finish = [&](int l) {
        if constexpr (PREC == 1) finish32<F16TAB>(tF, l, taps);
        else tmem_st1(tF + l, lerp_level(htaps));
      };
      const bool pre_k = pre && k < 8u;                               // levels 2k, 2k+1 of the next group ride in this query
      if (kPre && pre_k) pre_gather(2 * (int)k);
      if constexpr (TSHARED) {
        if constexpr (PREC == 0) h1_shared_h2(tA, P2h, reinterpret_cast<const uint32_t*>(s_Qt) + k * (kH / 2));
        else h1_shared_split(tA, P2, s_Qt + k * kH);
      } else {
        const float* tp = dir_of(fr.t, trow, k);
        h1_dir<PREC == 1>(tA, cw, [&](int q) { return P2s4[q * kRows]; }, __ldg(tp), __ldg(tp + 1), __ldg(tp + 2));
      }
      issue_layer<PREC, G>(c, 0, 2, 4, PREC == 1, 0, 3);
      if (kPre && pre_k) { pre_finish(2 * (int)k); pre_gather(2 * (int)k + 1); }
      if (TSHARED) {                                                  // shading factors: they do not need the MMA
        const float4 a = reinterpret_cast<const float4*>(s_Lt)[2 * k], d = reinterpret_cast<const float4*>(s_Lt)[2 * k + 1];
        L = make_float3(a.x, a.y, a.z); tpdf = a.w; tx = d.x; ty = d.y; tz = d.z;
      } else {
        const float* tp = dir_of(fr.t, trow, k);
        tx = __ldg(tp); ty = __ldg(tp + 1); tz = __ldg(tp + 2); tpdf = pdf_of(fr.t, trow, k);
        L = incoming(env, fr.t, trow, k, tx, ty, tz);
      }
      const float3 gg = brdf_cos_over_pdf(sp, bb, tx, ty, tz, -iwx, -iwy, -iwz, tpdf);
      wait_layer(c);
      if (kPre && pre_k) pre_finish(2 * (int)k + 1);
      const float v2 = vis_of(sp, PREC == 0 ? epi_fast(tD, cw) : epi_precise_v(tD, cw));
      lr = fmaf(v2 * L.x, gg.x, lr); lg = fmaf(v2 * L.y, gg.y, lg); lb = fmaf(v2 * L.z, gg.z, lb);
    }
    pre_done = pre;
    if (on) {
      float* a = acc + 4 * (owner & 0xFFu);
      atomicAdd(a, wr * lr); atomicAdd(a + 1, wgc * lg); atomicAdd(a + 2, wb * lb);
    }
  };

  // ---- tile loop (dynamic: work per tile varies with the number of occluded rays) ------------------------------------
  while (true) {
    if (c.t == 0) qctl[2] = (uint32_t)atomicAdd(counters, 1ull);
    wg_sync(c);
    const unsigned long long tile = qctl[2];
    if (__any_sync(0xFFFFFFFFu, tile >= ntiles)) break;      // WG-uniform; the vote tells the compiler so
    const unsigned long long tile_base = tile * kRows;
    const unsigned long long i_raw = tile_base + c.t;
    const bool valid = i_raw < fr.N;
    const unsigned long long i = valid ? i_raw : fr.N - 1;          // idle rows shadow the last point (uniform control flow)
    const bool live = valid && !(fr.mask && !fr.mask[i]);
    const float px = __ldg(fr.x + 3 * i), py = __ldg(fr.x + 3 * i + 1), pz = __ldg(fr.x + 3 * i + 2);
    const float ox = __ldg(fr.wo + 3 * i), oy = __ldg(fr.wo + 3 * i + 1), oz = __ldg(fr.wo + 3 * i + 2);
    float b[7];
    float r = 0.f, gch = 0.f, bch = 0.f;
    acc[4 * c.t] = 0.f; acc[4 * c.t + 1] = 0.f; acc[4 * c.t + 2] = 0.f;

    // ---- phase A: primary point ---------------------------------------------------------------------------------------
    const bool decode = !fr.brdf;
    encode_split_to<F16TAB, LIF>(tA, g, px, py, pz, (PREC == 1 && decode) ? Ps : nullptr);
    issue_layer<PREC, G>(c, 0, 0, 2, true, 0, 2);                     // P = W1f f + b1
    if (PREC == 1 && decode) {
      // fp32 model: the primary point's B runs in plain fp32 FFMAs (weights broadcast from L1) while the MMA is in
      // flight.  n = o/||o|| and n.w amplify an absolute error of o, and every sample of the pixel shares it, so the
      // 22-bit split arithmetic is not enough here; the cost is once per pixel.
      brdf_decode_scr<kRows>(sp, wts32, Ps, b);
    }
    wait_layer(c);
    // Ps (one float column per thread, used by brdf_decode_scr as its 64-entry scratch) and Ps4 (one float4 column per thread)
    // are two layouts of the SAME shared memory: a thread's float4 entries cover other threads' scratch entries.  Warps run
    // ahead of one another between barriers (warps 1-3 only bar.arrive in issue_layer), so every warp must have left
    // brdf_decode_scr before any warp stores P in the float4 layout -- without this barrier a fast warp corrupted a slow
    // warp's primary BRDF (or had its P overwritten) in about one frame out of ten: 32 pixels of one warp, errors up to 0.5.
    if (PREC == 1 && decode) wg_sync(c);
    store_D_f4(tD, Ps4);
    if (!decode) {
#pragma unroll
      for (int k = 0; k < 7; ++k) b[k] = __ldg(fr.brdf + i * 7 + k);
    } else if (PREC == 0) {
      brdf_primary<PREC, G>(c, cw, sp, b);                            // A columns 0..31 still hold f (hi | lo)
    }

    // ---- phase A2: direct term of Eq. 1 -------------------------------------------------------------------------------
    if ((fr.flags & 1u) && fr.d.S) {
      const uint32_t S = fr.d.S;
      float ar = 0.f, ag = 0.f, ab = 0.f;
      const float* dp = dir_of(fr.d, i, 0);
      float nx = __ldg(dp), ny = __ldg(dp + 1), nz = __ldg(dp + 2), np = pdf_of(fr.d, i, 0);
      for (uint32_t k = 0; k < S; ++k) {
        const float wx = nx, wy = ny, wz = nz, wp = np;
        const uint32_t k1 = k + 1 < S ? k + 1 : k;                    // prefetch the next direction
        dp = dir_of(fr.d, i, k1);
        nx = __ldg(dp); ny = __ldg(dp + 1); nz = __ldg(dp + 2); np = pdf_of(fr.d, i, k1);
        if (shadow) {
          h1_dir<PREC == 1>(tA, cw, [&](int q) { return Ps4[q * kRows]; }, wx, wy, wz);
          issue_layer<PREC, G>(c, 0, 2, 4, PREC == 1, 0, 3);
        }
        const float3 gg = brdf_cos_over_pdf(sp, b, wx, wy, wz, ox, oy, oz, wp);
        const float3 L = incoming(env, fr.d, i, k, wx, wy, wz);
        float vd = 1.f;
        if (shadow) {
          wait_layer(c);
          vd = vis_of(sp, PREC == 0 ? epi_fast(tD, cw) : epi_precise_v(tD, cw));
        }
        ar = fmaf(vd * L.x, gg.x, ar); ag = fmaf(vd * L.y, gg.y, ag); ab = fmaf(vd * L.z, gg.z, ab);
      }
      const float inv = 1.f / (float)S;
      r = ar * inv; gch = ag * inv; bch = ab * inv;
    }

    // ---- phases B + C: secondary rays -> work items -> L'_o -----------------------------------------------------------
    if constexpr (IND) if (S_i > 0) {
      const float wscale = 1.f / ((float)S_i * (float)S2);
      for (int j0 = 0; j0 < S_i; j0 += kChunkJ) {
        const int j1 = min(j0 + kChunkJ, S_i);
        for (int j = j0; j < j1; ++j) {
          const float* dp = dir_of(fr.s, i, j);
          const float wx = __ldg(dp), wy = __ldg(dp + 1), wz = __ldg(dp + 2), wp = pdf_of(fr.s, i, j);
          h1_dir<true>(tA, cw, [&](int q) { return Ps4[q * kRows]; }, wx, wy, wz);
          issue_layer<PREC, G>(c, 0, 2, 4, true, 0, 3);
          const float3 gg = brdf_cos_over_pdf(sp, b, wx, wy, wz, ox, oy, oz, wp);
          wait_layer(c);
          float zv, zt, v, t;
          epi_precise<false>(tD, cw, zv, zt);
          irt_maps(sp, zv, zt, v, t);
          const float m = (1.f - v) * wscale;
          const float gr = m * gg.x, ggc = m * gg.y, gb = m * gg.z;
          const bool push = live && (dense || gr != 0.f || ggc != 0.f || gb != 0.f);
          const unsigned bal = __ballot_sync(0xFFFFFFFFu, push);
          if (bal) {
            const int lane = threadIdx.x & 31, leader = __ffs(bal) - 1;
            uint32_t base = 0;
            if (lane == leader) base = atomicAdd(&qctl[1], (uint32_t)__popc(bal));
            base = __shfl_sync(0xFFFFFFFFu, base, leader);
            if (push) {
              float4* ip = reinterpret_cast<float4*>(myring + ((base + __popc(bal & ((1u << lane) - 1u))) & (kRing - 1)));
              __stcg(ip, make_float4(sec_hit(px, t, wx), sec_hit(py, t, wy), sec_hit(pz, t, wz), wx));
              __stcg(ip + 1, make_float4(wy, wz, gr, ggc));
              __stcg(ip + 2, make_float4(gb, __uint_as_float((uint32_t)c.t | ((uint32_t)j << 8)), 0.f, 0.f));
            }
          }
          n_rays += live ? 1u : 0u;
        }
        wg_sync(c);                                                   // items of this chunk are visible to the whole WG
        uint32_t count = qctl[1] - head;
        const bool last = j1 == S_i;
        while (__any_sync(0xFFFFFFFFu, count >= (uint32_t)kRows || (last && count > 0u))) {
          const uint32_t n = count < (uint32_t)kRows ? count : (uint32_t)kRows;
          const uint32_t rest = count - n;                            // the group after this one, if it will be drained next
          const uint32_t nn = (rest >= (uint32_t)kRows || (last && rest > 0u)) ? (rest < (uint32_t)kRows ? rest : (uint32_t)kRows) : 0u;
          drain_group(n, tile_base, nn);
          head += n; count -= n;
          n_items += (uint32_t)c.t < n ? 1u : 0u;
        }
      }
      wg_sync(c);                                                     // every contribution has landed in acc
      r += acc[4 * c.t]; gch += acc[4 * c.t + 1]; bch += acc[4 * c.t + 2];
    }
    if (valid) {
      rgb[3 * i] = live ? r : 0.f; rgb[3 * i + 1] = live ? gch : 0.f; rgb[3 * i + 2] = live ? bch : 0.f;
    }
  }
  // ---- teardown ---------------------------------------------------------------------------------------------------------
  for (int o = 16; o > 0; o >>= 1) {
    n_items += __shfl_xor_sync(0xFFFFFFFFu, n_items, o);
    n_rays += __shfl_xor_sync(0xFFFFFFFFu, n_rays, o);
  }
  if ((threadIdx.x & 31) == 0 && (n_items | n_rays)) { atomicAdd(counters + 1, (unsigned long long)n_items); atomicAdd(counters + 2, (unsigned long long)n_rays); }
  fence_before();
  __syncthreads();
  if (warp == 0) {
    fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*s_tmem), "r"(512u) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------- trace kernel
// hashrender_trace with the encode fused (a1-a4, a6, a7) for fp16 models -- the kernel of the encode + IRT sweep
// (BASELINE.json configs[4]).  Same warpgroup scheme with G = 4.  t is an output, so the fp32 epilogue is used (features hi/lo
// split for P, fp16 h1).  Levels whose gathers are in flight together: two, and one in the instantiation for tables far beyond
// the L2 (HINT).  Measured at 2^24 points with the cell-major levels (ms at T = 2^16 / 2^19 / 2^22 / 2^24): one level 4.36 / 4.80 /
// 8.73 / 9.25, two 4.31 / 4.70 / 8.57 / 9.53, four 4.46 / 4.92 / 8.83 / 9.48.  (Before the cell-major levels four was best:
// 16 warps x 32 outstanding loads; a cell-major level is one load, so four levels no longer means 32.)
// With the paired loads of the L2-resident fp16 tables (6 loads per level, MODE 2) four levels are best again: T = 2^16 4.12 -> 4.07,
// 2^19 4.65 -> 4.52 (same box).
constexpr int kTraceG = 4;
#ifdef HR_TRACE_LIF
constexpr int kTraceLIF = HR_TRACE_LIF, kTraceLIFHint = HR_TRACE_LIF, kTraceLIFRes = HR_TRACE_LIF;
#else
constexpr int kTraceLIF = 2, kTraceLIFHint = 1, kTraceLIFRes = 4;
#endif
template <int PREC> constexpr size_t trace_smem() {
  return 1024 + (size_t)kHiTileBytes * (PREC ? 2 : 1) + kOnesBytes + (size_t)kTraceG * kH * kRows * 4 + 8 * kMaxG + 16;
}

// caller-supplied features f[2 L] (fp32) -> A columns 0..15 (hi) | 16..31 (lo), as encode_split_to leaves them
template <int LIF>
__device__ __forceinline__ void feat_split_to(uint32_t tA, const GridP& g, const float* __restrict__ f) {
#pragma unroll 1
  for (int l0 = 0; l0 < kMaxL; l0 += LIF) {
    uint32_t hi[LIF], lo[LIF];
#pragma unroll
    for (int q = 0; q < LIF; ++q) {
      hi[q] = 0u; lo[q] = 0u;
      if (l0 + q < (int)g.L) {
        const float2 v = __ldg(reinterpret_cast<const float2*>(f) + l0 + q);
        split_pair(v.x, v.y, hi[q], lo[q]);
      }
    }
    tmem_stN(tA + l0, hi);
    tmem_stN(tA + 16 + l0, lo);
  }
}

// PREC = 0: fp16 models (fp16 h1, one MMA pass).  PREC = 1: fp32 models in hi/lo split precision -- exactly the arithmetic
// k_render_wg<PREC = 1> runs for its direct / secondary queries (h1_dir<true>, three passes, epi_precise), so hashrender_trace
// on an fp32 model checks z_v, t, x' of the production path stage by stage.  feat != nullptr: the caller's features replace H(x).
// MODE 0: tables beyond the L2; 1: far beyond it (L2 policies on the gathers); 2: L2-resident fp16 tables (paired loads)
template <bool F16TAB, int PREC, int MODE = 0>
__global__ void __launch_bounds__(kRows* kTraceG, 1)
    k_trace_wg(const __grid_constant__ GridP g, ShadeP sp, const __grid_constant__ TcConst cw, const uint8_t* __restrict__ wtiles,
               const float* __restrict__ x, const float* __restrict__ feat, unsigned long long N, DirsetP ds, float* __restrict__ vis,
               float* __restrict__ zvo, float* __restrict__ to, float* __restrict__ xsec) {
  constexpr int G = kTraceG;
  using CL = Cols<PREC, G>;
  constexpr int kTiles = kHiTileBytes * (PREC ? 2 : 1);
  extern __shared__ uint8_t smem_raw[];
  uint8_t* s_tiles = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  uint8_t* s_ones = s_tiles + kTiles;
  float4* s_P = reinterpret_cast<float4*>(s_ones + kOnesBytes);
  uint64_t* s_mbar = reinterpret_cast<uint64_t*>(s_P + (size_t)G * (kH / 4) * kRows);
  uint32_t* s_tmem = reinterpret_cast<uint32_t*>(s_mbar + kMaxG);
  const int wgi = threadIdx.x / kRows, warp = threadIdx.x >> 5;
  WgCtx c;
  c.t = threadIdx.x % kRows;
  c.bar_id = 1 + wgi;
  c.rot = 0; c.rot_mask = 0u;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (threadIdx.x < G) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(s_mbar + threadIdx.x)) : "memory");
  if (threadIdx.x == 0) asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  {
    const uint4* src = reinterpret_cast<const uint4*>(wtiles);
    uint4* dst = reinterpret_cast<uint4*>(s_tiles);
    for (int i = threadIdx.x; i < kTiles / 16; i += kRows * G) dst[i] = __ldg(src + i);
  }
  fill_ones(s_ones, kRows * G);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  fence_before();
  __syncthreads();
  fence_after();
  // warp-uniform by construction; the reductions tell the compiler so, which keeps the MMA operands (TMEM addresses, smem
  // descriptors, the mbarrier) in uniform registers instead of re-broadcasting them from a lane before every tcgen05.mma
  c.tmem = __reduce_min_sync(0xFFFFFFFFu, *s_tmem + CL::stride * wgi);
  c.lane = __reduce_min_sync(0xFFFFFFFFu, (uint32_t)((warp & 3) * 32) << 16);     // tcgen05.ld / st addresses are uniform operands too
  c.mbar = __reduce_min_sync(0xFFFFFFFFu, smem_u32(s_mbar + wgi));
  c.phase = 0;
  c.tile0 = smem_u32(s_tiles);
  c.lo_off = kHiTileBytes;
  c.ones = smem_u32(s_ones);
  const uint32_t tA = c.tmem + c.lane, tD = c.tmem + c.lane + CL::d;
  float4* Ps4 = s_P + (size_t)wgi * (kH / 4) * kRows + c.t;
  const unsigned long long ntiles = (N + kRows - 1) / kRows;
  const uint32_t D = g.L * 2u;
  L2Pol pol;
  constexpr bool HINT = MODE == 1;
  if constexpr (HINT) pol = make_l2pol();
  for (unsigned long long tile = (unsigned long long)blockIdx.x * G + wgi; tile < ntiles; tile += (unsigned long long)gridDim.x * G) {
    const unsigned long long i_raw = tile * kRows + c.t;
    const bool valid = i_raw < N;
    const unsigned long long i = valid ? i_raw : N - 1;
    float px = 0.f, py = 0.f, pz = 0.f;
    if (x) { px = __ldg(x + 3 * i); py = __ldg(x + 3 * i + 1); pz = __ldg(x + 3 * i + 2); }
    if (feat) feat_split_to<4>(tA, g, feat + i * D);
    else if constexpr (HINT) encode_split_to<F16TAB, kTraceLIFHint, 0>(tA, g, px, py, pz, nullptr, &pol);
    else if constexpr (MODE == 2) encode_split_to<F16TAB, kTraceLIFRes, 1>(tA, g, px, py, pz);
    else encode_split_to<F16TAB, kTraceLIF>(tA, g, px, py, pz);
    issue_layer<PREC, G>(c, 0, 0, 2, true, 0, 2);                     // P = W1f f + b1, split-precision f
    wait_layer(c);
    store_D_f4(tD, Ps4);
    for (uint32_t sidx = 0; sidx < ds.S; ++sidx) {
      const float* dp = dir_of(ds, i, sidx);
      const float wx = __ldg(dp), wy = __ldg(dp + 1), wz = __ldg(dp + 2);
      h1_dir<PREC == 1>(tA, cw, [&](int q) { return Ps4[q * kRows]; }, wx, wy, wz);
      issue_layer<PREC, G>(c, 0, 2, 4, PREC == 1, 0, 3);
      wait_layer(c);
      float zv, zt, v, t;
      epi_precise<false>(tD, cw, zv, zt);
      irt_maps(sp, zv, zt, v, t);
      if (valid) {
        const unsigned long long o = i * ds.S + sidx;
        vis[o] = v; to[o] = t;
        if (zvo) zvo[o] = zv;
        if (xsec) { xsec[o * 3] = sec_hit(px, t, wx); xsec[o * 3 + 1] = sec_hit(py, t, wy); xsec[o * 3 + 2] = sec_hit(pz, t, wz); }
      }
    }
  }
  fence_before();
  __syncthreads();
  if (warp == 0) {
    fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*s_tmem), "r"(512u) : "memory");
  }
}

template <bool F16TAB, int PREC>
inline cudaError_t launch_trace_one(const GridP& g, const ShadeP& sp, const TcConst& cw, const uint8_t* d_tiles, const float* x,
                                    const float* feat, unsigned long long N, const DirsetP& ds, float* vis, float* zv, float* t,
                                    float* xsec, int num_sms, cudaStream_t st) {
  const unsigned long long need = ((N + kRows - 1) / kRows + kTraceG - 1) / kTraceG;
  const int grid = (int)(need < (unsigned long long)num_sms ? need : (unsigned long long)num_sms);
  if (F16TAB && g.l2_hint && !feat)
    k_trace_wg<F16TAB, PREC, F16TAB ? 1 : 0><<<grid, kRows * kTraceG, trace_smem<PREC>(), st>>>(g, sp, cw, d_tiles, x, feat, N, ds, vis, zv, t, xsec);
  else if (F16TAB && g.pair_loads && !feat)
    k_trace_wg<F16TAB, PREC, F16TAB ? 2 : 0><<<grid, kRows * kTraceG, trace_smem<PREC>(), st>>>(g, sp, cw, d_tiles, x, feat, N, ds, vis, zv, t, xsec);
  else
    k_trace_wg<F16TAB, PREC><<<grid, kRows * kTraceG, trace_smem<PREC>(), st>>>(g, sp, cw, d_tiles, x, feat, N, ds, vis, zv, t, xsec);
  return cudaGetLastError();
}
// the opt-in to > 48 KB of dynamic shared memory is per device: hashrender_create calls this for the handle's device
template <bool F16TAB, int PREC>
inline cudaError_t trace_attr() {
  cudaError_t e = cudaFuncSetAttribute(k_trace_wg<F16TAB, PREC, F16TAB ? 1 : 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)trace_smem<PREC>());
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(k_trace_wg<F16TAB, PREC, F16TAB ? 2 : 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)trace_smem<PREC>());
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(k_trace_wg<F16TAB, PREC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)trace_smem<PREC>());
}

// ---------------------------------------------------------------------------------------------------- host side
// Blob = [ TcConst | hi tiles (34 KB) | lo tiles (34 KB) ].  hi = fp16(w), lo = fp16(w - hi); bias K-steps only in the hi tiles.
inline void prepare_weights(const hr_config& cfg, const float* bw, const float* iw, std::vector<uint8_t>& out) {
  std::vector<uint8_t> hi;
  tc::prepare_weights(cfg, bw, iw, hi);                 // TcConst + hi tiles (weights rounded to fp16, biases split)
  out.assign(sizeof(TcConst) + 2 * kHiTileBytes, 0);
  memcpy(out.data(), hi.data(), sizeof(TcConst) + kHiTileBytes);
  const int D = cfg.L * cfg.F, H = kH, Din = D + 3;
  uint8_t* lo = out.data() + sizeof(TcConst) + kHiTileBytes;
  auto put_lo = [&](int t, int j, int k, float v) {
    const float h = __half2float(__float2half_rn(v));
    *reinterpret_cast<__half*>(lo + (size_t)t * kTileBytes + tile_off(j, k)) = __float2half_rn(v - h);
  };
  const float* BW1 = bw; const float* BW2 = BW1 + H * D + H; const float* BW3 = BW2 + H * H + H;
  const float* IW1 = iw; const float* IW2 = IW1 + H * Din + H;
  for (int j = 0; j < H; ++j) {
    for (int k = 0; k < D; ++k) { put_lo(0, j, k, IW1[j * Din + k]); put_lo(1, j, k, BW1[j * D + k]); }
    for (int k = 0; k < H; ++k) { put_lo(2, j, k, IW2[j * H + k]); put_lo(3, j, k, BW2[j * H + k]); }
    for (int q = 0; q < 7; ++q) put_lo(4, q, j, BW3[q * H + j]);
  }
}

inline bool frame_supported(const FrameP& fr) { return !(fr.flags & 4u) || fr.t.stride != 0 || fr.t.S <= (uint32_t)kMaxS2; }

template <bool F16TAB, int PREC, bool TSHARED, int G, bool IND = true>
inline cudaError_t launch_one(const GridP& g, const EnvP& env, const ShadeP& sp, const TcConst& cw, const uint8_t* d_tiles,
                              const float* wts32, const FrameP& fr, float* rgb, Item* ring, unsigned long long* counters, int num_sms, cudaStream_t st) {
  using SP = SmemPlan<PREC, TSHARED, G>;
  auto kern = k_render_wg<F16TAB, PREC, TSHARED, G, IND>;
  cudaError_t e = cudaMemsetAsync(counters, 0, 8, st);                // the tile counter; the statistics keep accumulating
  if (e != cudaSuccess) return e;
  const unsigned long long tiles = (fr.N + kRows - 1) / kRows;
  const unsigned long long need = (tiles + G - 1) / G;
  const int grid = (int)(need < (unsigned long long)num_sms ? need : (unsigned long long)num_sms);
  kern<<<grid, kRows * G, SP::bytes, st>>>(g, env, sp, cw, d_tiles, wts32, fr, rgb, ring, counters);
  return cudaGetLastError();
}

template <bool F16TAB, int PREC, bool TSHARED, int G, bool IND = true>
inline cudaError_t render_attr() {
  return cudaFuncSetAttribute(k_render_wg<F16TAB, PREC, TSHARED, G, IND>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)SmemPlan<PREC, TSHARED, G>::bytes);
}

}  // namespace wg
}  // namespace hr
