// hr_gnet.cuh -- device side of the CNN direct-illumination renderer G (Q45-Q51), the step
// that produces the hash-grid renderer's inputs (x, n, a, r, mask).
//
// Every convolution is ONE kernel, k_gconv: an implicit GEMM on tcgen05 with both operands staged by TMA.
//   A = activations, fp16, NHWC.  A 1x1 layer sees the image as a flat [pixels][K] matrix (2-D tensor map, 128 consecutive pixels
//       per tile); a 3x3 layer sees a zero-bordered [H+2][W+2][K] tensor (3-D tensor map) and a tile is a 16-row x 8-pixel patch
//       of the output, so tap (ky, kx) of the filter is the SAME box shifted by (ky, kx): nine TMA loads per K-chunk, no im2col.
//       Either way a stage is 128 rows x 64 channels = 128 B rows in SWIZZLE_128B, exactly the K-major UMMA operand tile.
//   B = weights [Cout][taps * K], K-major, one [Cout x 64] box per stage.
//   D = 128 x Cout fp32 accumulator in TMEM, double-buffered (2 x Cout <= 512 columns): the epilogue of tile i (TMEM -> registers,
//       + bias, fp32 store, per-channel sum / sum of squares for the instance norm) overlaps the MMAs of tile i + 1.
// Warp roles: warp 0 = TMA producer, warp 1 = MMA issuer, warps 2..5 = epilogue (one TMEM lane quarter each).
//
// Precision (Q51): the network amplifies a perturbation of its activations about a hundredfold over its 34 layers, so
// fp16 activations cannot hold even 3e-3.  Activations are therefore carried as hi + lo fp16 pairs (K = [hi | lo], the weight
// chunk is used for both halves: two MMA passes, fp32 accumulate), weights are fp16-representable (rounded once by the caller's
// generator), and everything between two convolutions (instance norm, GELU, residual sum, bilinear upsampling) is fp32.
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "hr_kernels_tc.cuh"

namespace hr {
namespace gn {
using namespace hr::tc;

constexpr int kStages = 4;
constexpr int kABytes = 128 * 128;                 // 128 rows x 64 fp16
constexpr int kBBytes = 256 * 128;                 // up to 256 output channels x 64 fp16
constexpr int kStageBytes = kABytes + kBBytes;
constexpr size_t kConvSmem = 1024 + (size_t)kStages * kStageBytes + 2 * 256 * 8 + 256;
constexpr int kOutCh = 11;                         // n3 a3 r1 x3 mask1

struct ConvP {
  int taps;               // 1 or 9
  int kchunks;            // 64-channel chunks of the activation tensor per tap (hi and lo halves together)
  int wchunks;            // 64-channel chunks of the weight tensor per tap (= kchunks / 2: the lo half re-uses the hi half's weights)
  int Cout;
  int H, W;               // output image
  long long N;            // H * W
  int tiles_x, tiles;
  const float* bias;      // [Cout]
  float* pre;             // [N][Cout] fp32, convolution output before the norm
  double* stats;          // [2][Cout]: sum, sum of squares over the image (zeroed before the launch)
};

// ---- PTX wrappers the render kernels do not need --------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t mbar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory"); }
__device__ __forceinline__ void mbar_wait1(uint32_t mbar, uint32_t parity) {        // one thread (or a whole warp) waits
  asm volatile(
      "{\n\t.reg .pred P1;\n\tLAB_WAIT:\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, 0x989680;\n\t@P1 bra DONE;\n\tbra LAB_WAIT;\n\tDONE:\n\t}\n" ::"r"(mbar),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, uint32_t mbar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst), "l"(tm), "r"(c0),
               "r"(c1), "r"(mbar)
               : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, uint32_t mbar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst), "l"(tm),
               "r"(c0), "r"(c1), "r"(c2), "r"(mbar)
               : "memory");
}
__device__ __forceinline__ uint32_t idesc_n(int N) { return (1u << 4) | ((uint32_t)(N >> 3) << 17) | ((128u >> 4) << 24); }

// Sum over the 32 lanes of a warp of 32 per-lane values, one value per channel: recursive halving, 31 shuffles; lane l ends up with
// the total of channel l.
__device__ __forceinline__ float lanes_reduce32(float (&v)[32], int lane) {
#pragma unroll
  for (int off = 16; off >= 1; off >>= 1) {
    const bool up = lane & off;
#pragma unroll
    for (int j = 0; j < off; ++j) {
      const float send = up ? v[j] : v[j + off];
      const float keep = up ? v[j + off] : v[j];
      v[j] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, off);
    }
  }
  return v[0];
}

// ---------------------------------------------------------------------------------------------------- the convolution
template <int TAPS>
__global__ void __launch_bounds__(192, 1)
    k_gconv(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, ConvP p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
  // per-CTA statistics in double: the order in which the epilogue warps (and, below, the CTAs) add their partial sums then
  // changes the result only at the 1e-16 level, so the instance norm -- and with it the whole forward pass, which amplifies a 1e-7
  // perturbation of a normalised map to 5e-5 at the output -- is reproducible run to run
  double* s_sum = reinterpret_cast<double*>(base + (size_t)kStages * kStageBytes);
  double* s_sq = s_sum + 256;
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(s_sq + 256);          // full[kStages], empty[kStages], tfull[2], tempty[2]
  uint32_t* s_tmem = reinterpret_cast<uint32_t*>(s_bar + 2 * kStages + 4);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t bar0 = smem_u32(s_bar);
  auto full = [&](int s) { return bar0 + 8u * s; };
  auto empty = [&](int s) { return bar0 + 8u * (kStages + s); };
  auto tfull = [&](int a) { return bar0 + 8u * (2 * kStages + a); };
  auto tempty = [&](int a) { return bar0 + 8u * (2 * kStages + 2 + a); };

  for (int i = threadIdx.x; i < 512; i += blockDim.x) s_sum[i] = 0.0;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s_tmem)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (threadIdx.x == 32) {
    for (int s = 0; s < kStages; ++s) { mbar_init(full(s), 1); mbar_init(empty(s), 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(tfull(a), 1); mbar_init(tempty(a), 128); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem = *s_tmem;
  const int iters = p.taps * p.kchunks;
  const uint32_t a0 = smem_u32(base), stage_bytes = (uint32_t)p.Cout * 128u + kABytes;

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      uint32_t s = 0, ph = 0;
      for (int tile = blockIdx.x; tile < p.tiles; tile += gridDim.x) {
        const int tx = tile % p.tiles_x, ty = tile / p.tiles_x;
        for (int it = 0; it < iters; ++it) {
          mbar_wait1(empty(s), ph ^ 1u);
          mbar_expect_tx(full(s), stage_bytes);
          const int tap = it / p.kchunks, kc = it - tap * p.kchunks;
          const uint32_t dstA = a0 + s * kStageBytes, dstB = dstA + kABytes;
          if (TAPS == 9) tma_load_3d(dstA, &tmA, kc * 64, tx * 8 + tap % 3, ty * 16 + tap / 3, full(s));
          else tma_load_2d(dstA, &tmA, kc * 64, tile * 128, full(s));
          tma_load_2d(dstB, &tmB, (tap * p.wchunks + kc % p.wchunks) * 64, 0, full(s));
          if (++s == kStages) { s = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer (whole warp converged, one elected lane issues) =====
    uint32_t s = 0, ph = 0, acc = 0, aph = 0;
    const uint32_t idesc = idesc_n(p.Cout);
    for (int tile = blockIdx.x; tile < p.tiles; tile += gridDim.x) {
      mbar_wait(tempty(acc), aph ^ 1u);
      fence_after();
      const uint32_t d = tmem + acc * (uint32_t)p.Cout;
      for (int it = 0; it < iters; ++it) {
        mbar_wait(full(s), ph);
        fence_after();
        const uint64_t da = make_bdesc(a0 + s * kStageBytes), db = make_bdesc(a0 + s * kStageBytes + kABytes);
#pragma unroll
        for (int k = 0; k < 4; ++k) mma_f16_ss_elect(d, da + 2 * k, db + 2 * k, idesc, (it | k) ? 1u : 0u);
        mma_commit_elect(empty(s));
        if (++s == kStages) { s = 0; ph ^= 1u; }
      }
      mma_commit_elect(tfull(acc));
      if (++acc == 2) { acc = 0; aph ^= 1u; }
    }
  } else {
    // ===== epilogue: TMEM -> registers -> (+ bias) fp32 store, per-channel statistics =====
    const int q = warp & 3;                                       // TMEM lane quarter this warp may read
    const int row = q * 32 + lane;
    uint32_t acc = 0, aph = 0;
    for (int tile = blockIdx.x; tile < p.tiles; tile += gridDim.x) {
      long long pix;
      bool valid;
      if (TAPS == 9) {
        const int tx = tile % p.tiles_x, ty = tile / p.tiles_x;
        const int y = ty * 16 + (row >> 3), x = tx * 8 + (row & 7);
        valid = y < p.H && x < p.W;
        pix = (long long)y * p.W + x;
      } else {
        pix = (long long)tile * 128 + row;
        valid = pix < p.N;
      }
      mbar_wait(tfull(acc), aph);
      fence_after();
      const uint32_t t0 = tmem + acc * (uint32_t)p.Cout + ((uint32_t)(q * 32) << 16);
      for (int c0 = 0; c0 < p.Cout; c0 += 32) {
        uint32_t r[32];
        tmem_ld32(t0 + c0, r);
        wait_ld();
        float v[32], w[32];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float4 b4 = __ldg(reinterpret_cast<const float4*>(p.bias + c0) + j);
          v[4 * j] = __uint_as_float(r[4 * j]) + b4.x; v[4 * j + 1] = __uint_as_float(r[4 * j + 1]) + b4.y;
          v[4 * j + 2] = __uint_as_float(r[4 * j + 2]) + b4.z; v[4 * j + 3] = __uint_as_float(r[4 * j + 3]) + b4.w;
        }
        if (valid) {
          float4* o = reinterpret_cast<float4*>(p.pre + pix * p.Cout + c0);
#pragma unroll
          for (int j = 0; j < 8; ++j) o[j] = make_float4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
        }
#pragma unroll
        for (int j = 0; j < 32; ++j) { v[j] = valid ? v[j] : 0.f; w[j] = v[j] * v[j]; }
        const float sum = lanes_reduce32(v, lane), sq = lanes_reduce32(w, lane);
        atomicAdd(s_sum + c0 + lane, (double)sum);
        atomicAdd(s_sq + c0 + lane, (double)sq);
      }
      fence_before();
      mbar_arrive(tempty(acc));
      if (++acc == 2) { acc = 0; aph ^= 1u; }
    }
  }
  fence_before();
  __syncthreads();
  for (int c = threadIdx.x; c < p.Cout; c += blockDim.x) {
    atomicAdd(p.stats + c, s_sum[c]);
    atomicAdd(p.stats + p.Cout + c, s_sq[c]);
  }
  if (warp == 0) {
    fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------- element-wise stages
__device__ __forceinline__ float gelu_f(float x) { return 0.5f * x * (1.f + erff(x * 0.70710678118654752f)); }
// value -> (hi, lo) fp16 with hi + lo = v to 2^-22
__device__ __forceinline__ void split16(float v, __half& hi, __half& lo) {
  hi = __float2half_rn(v);
  lo = __float2half_rn(v - __half2float(hi));
}

struct NormP {
  const float* pre;        // [N][C]
  const double* stats;     // [2][C]
  const float* gamma; const float* beta;
  float* res;              // residual stream [N][C] (mode-dependent)
  float* feat;             // fp32 feature output [N][C] (mode 3)
  __half* act;             // fp16 hi|lo activation tensor for the next convolution
  long long N; int C, H, W;
  int mode;                // 0: res = y, act = split(y) (stem)   1: act = split(y) (first layer of a residual block)
                           // 2: res += y, act = split(res) (second layer)   3: feat = y   4: act (zero-bordered [H+2][W+2][2C]) = split(y)
};

// y = GELU(IN(pre)): one thread per (pixel, 8 channels); the per-channel scale / shift come from the image statistics
__global__ void __launch_bounds__(256) k_gnorm(NormP p) {
  extern __shared__ float s_ab[];                         // a[C], b[C]: y_norm = x a + b
  for (int c = threadIdx.x; c < p.C; c += blockDim.x) {
    const double m = p.stats[c] / (double)p.N;
    double var = p.stats[p.C + c] / (double)p.N - m * m;
    var = var > 0.0 ? var : 0.0;
    const double rstd = 1.0 / sqrt(var + 1e-5);
    const double a = rstd * (double)p.gamma[c];
    s_ab[c] = (float)a;
    s_ab[p.C + c] = (float)((double)p.beta[c] - m * a);
  }
  __syncthreads();
  // 32-bit index arithmetic (the host refuses images with 2^31 or more (pixel, 8-channel) groups): 64-bit divisions cost more
  // than the GELU
  const uint32_t groups = (uint32_t)p.C / 8u;
  const uint32_t total = (uint32_t)p.N * groups;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
    const uint32_t pixu = i / groups;
    const long long pix = pixu;
    const int c0 = (int)(i - pixu * groups) * 8;
    const float4 x0 = *reinterpret_cast<const float4*>(p.pre + pix * p.C + c0), x1 = *reinterpret_cast<const float4*>(p.pre + pix * p.C + c0 + 4);
    float v[8] = {x0.x, x0.y, x0.z, x0.w, x1.x, x1.y, x1.z, x1.w};
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = gelu_f(fmaf(v[j], s_ab[c0 + j], s_ab[p.C + c0 + j]));
    if (p.mode == 3) {
      float4* o = reinterpret_cast<float4*>(p.feat + pix * p.C + c0);
      o[0] = make_float4(v[0], v[1], v[2], v[3]); o[1] = make_float4(v[4], v[5], v[6], v[7]);
      continue;
    }
    if (p.mode == 0 || p.mode == 2) {
      float4* rp = reinterpret_cast<float4*>(p.res + pix * p.C + c0);
      if (p.mode == 2) {
        const float4 r0 = rp[0], r1 = rp[1];
        v[0] += r0.x; v[1] += r0.y; v[2] += r0.z; v[3] += r0.w; v[4] += r1.x; v[5] += r1.y; v[6] += r1.z; v[7] += r1.w;
      }
      rp[0] = make_float4(v[0], v[1], v[2], v[3]); rp[1] = make_float4(v[4], v[5], v[6], v[7]);
    }
    __align__(16) __half hi[8], lo[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) split16(v[j], hi[j], lo[j]);
    long long row = pix;
    if (p.mode == 4) { const uint32_t y = pixu / (uint32_t)p.W, x = pixu - y * (uint32_t)p.W; row = (long long)(y + 1) * (p.W + 2) + x + 1; }
    __half* o = p.act + row * (2 * p.C) + c0;
    *reinterpret_cast<uint4*>(o) = *reinterpret_cast<const uint4*>(hi);
    *reinterpret_cast<uint4*>(o + p.C) = *reinterpret_cast<const uint4*>(lo);
  }
}

// gamma = [o, d] rays [N][6] fp32 -> fp16 hi|lo in channels 0..5 | 6..11 of a [N][64] tensor (the other channels stay zero)
__global__ void __launch_bounds__(256) k_grays(const float* __restrict__ rays, __half* __restrict__ act, long long N) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N * 6; i += (long long)gridDim.x * blockDim.x) {
    const long long pix = i / 6; const int c = (int)(i - pix * 6);
    __half hi, lo;
    split16(rays[i], hi, lo);
    act[pix * 64 + c] = hi; act[pix * 64 + 6 + c] = lo;
  }
}

// bilinear x2 (align_corners = false: output pixel j samples the input at (j + 0.5)/2 - 0.5, clamped to the border) of an fp32
// [h][w][C] map into the zero-bordered fp16 hi|lo tensor [2h+2][2w+2][2C] the next 3x3 convolution reads
__device__ __forceinline__ void up_taps(int j, int n, int& i0, int& i1, float& f) {
  const float s = fmaxf((j + 0.5f) * 0.5f - 0.5f, 0.f);
  i0 = (int)s; i1 = min(i0 + 1, n - 1); f = s - (float)i0;
}
__global__ void __launch_bounds__(256) k_gupsample(const float* __restrict__ in, __half* __restrict__ act, int h, int w, int C) {
  const int H = 2 * h, W = 2 * w;
  const uint32_t groups = (uint32_t)C / 8u, total = (uint32_t)H * (uint32_t)W * groups;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
    const uint32_t pix = i / groups;
    const int c0 = (int)(i - pix * groups) * 8;
    const int y = (int)(pix / (uint32_t)W), x = (int)(pix - (uint32_t)y * (uint32_t)W);
    int y0, y1, x0, x1; float fy, fx;
    up_taps(y, h, y0, y1, fy); up_taps(x, w, x0, x1, fx);
    const float* p00 = in + ((long long)y0 * w + x0) * C + c0; const float* p01 = in + ((long long)y0 * w + x1) * C + c0;
    const float* p10 = in + ((long long)y1 * w + x0) * C + c0; const float* p11 = in + ((long long)y1 * w + x1) * C + c0;
    __align__(16) __half hi[8], lo[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const float top = p00[j] * (1.f - fx) + p01[j] * fx, bot = p10[j] * (1.f - fx) + p11[j] * fx;
      split16(top * (1.f - fy) + bot * fy, hi[j], lo[j]);
    }
    __half* o = act + ((long long)(y + 1) * (W + 2) + x + 1) * (2 * C) + c0;
    *reinterpret_cast<uint4*>(o) = *reinterpret_cast<const uint4*>(hi);
    *reinterpret_cast<uint4*>(o + C) = *reinterpret_cast<const uint4*>(lo);
  }
}

// "output mapping" 1x1 convolution of an SR block (PAPER.md:68b) + the output skip (PAPER.md:68a): maps = W f + b + up2(previous
// maps).  The last block also applies the output maps (Q50) and writes the arrays hr_frame takes.
struct MapP {
  const float* feat;       // [H][W][C]
  const float* Wm;         // [11][C]
  const float* bm;         // [11]
  const float* prev;       // [H/2][W/2][11] or nullptr
  float* out;              // [H][W][11]
  int H, W, C;
  float* x; float* brdf; uint8_t* mask;      // final arrays (nullable)
  float rough_min;
};
__global__ void __launch_bounds__(128) k_gmap(MapP p) {
  extern __shared__ float s_w[];                          // [11][C] + [11]
  for (int i = threadIdx.x; i < kOutCh * p.C + kOutCh; i += blockDim.x) s_w[i] = i < kOutCh * p.C ? p.Wm[i] : p.bm[i - kOutCh * p.C];
  __syncthreads();
  const uint32_t N = (uint32_t)p.H * (uint32_t)p.W;
  for (uint32_t pix = blockIdx.x * blockDim.x + threadIdx.x; pix < N; pix += gridDim.x * blockDim.x) {
    float o[kOutCh];
#pragma unroll
    for (int k = 0; k < kOutCh; ++k) o[k] = s_w[kOutCh * p.C + k];
    const float4* f = reinterpret_cast<const float4*>(p.feat + (size_t)pix * p.C);
    for (int c = 0; c < p.C / 4; ++c) {
      const float4 v = f[c];
#pragma unroll
      for (int k = 0; k < kOutCh; ++k) {
        const float* wr = s_w + k * p.C + 4 * c;
        o[k] = fmaf(v.x, wr[0], fmaf(v.y, wr[1], fmaf(v.z, wr[2], fmaf(v.w, wr[3], o[k]))));
      }
    }
    if (p.prev) {
      const int y = (int)(pix / (uint32_t)p.W), x = (int)(pix - (uint32_t)y * (uint32_t)p.W), h = p.H / 2, w = p.W / 2;
      int y0, y1, x0, x1; float fy, fx;
      up_taps(y, h, y0, y1, fy); up_taps(x, w, x0, x1, fx);
      const float* p00 = p.prev + ((long long)y0 * w + x0) * kOutCh; const float* p01 = p.prev + ((long long)y0 * w + x1) * kOutCh;
      const float* p10 = p.prev + ((long long)y1 * w + x0) * kOutCh; const float* p11 = p.prev + ((long long)y1 * w + x1) * kOutCh;
#pragma unroll
      for (int k = 0; k < kOutCh; ++k) {
        const float top = p00[k] * (1.f - fx) + p01[k] * fx, bot = p10[k] * (1.f - fx) + p11[k] * fx;
        o[k] += top * (1.f - fy) + bot * fy;
      }
    }
    if (p.out) {
#pragma unroll
      for (int k = 0; k < kOutCh; ++k) p.out[(size_t)pix * kOutCh + k] = o[k];
    }
    if (p.brdf) {
      const float inv = 1.f / fmaxf(sqrtf(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]), 1e-12f);
      float* b = p.brdf + (size_t)pix * 7;
      b[0] = o[0] * inv; b[1] = o[1] * inv; b[2] = o[2] * inv;
      b[3] = sigmoidf_(o[3]); b[4] = sigmoidf_(o[4]); b[5] = sigmoidf_(o[5]);
      b[6] = p.rough_min + (1.f - p.rough_min) * sigmoidf_(o[6]);
    }
    if (p.x) { float* xo = p.x + (size_t)pix * 3; xo[0] = sigmoidf_(o[7]); xo[1] = sigmoidf_(o[8]); xo[2] = sigmoidf_(o[9]); }
    if (p.mask) p.mask[pix] = o[10] > 0.f ? 1 : 0;
  }
}

}  // namespace gn
}  // namespace hr
