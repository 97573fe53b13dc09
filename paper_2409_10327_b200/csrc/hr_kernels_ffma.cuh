// hr_kernels_ffma.cuh -- fp32 FFMA implementation of every step a1-a11 (exact-fp32 path: mlp_dtype == HR_F32,
// and the parity baseline for the tensor-core path).  One thread owns one point and walks its direction sets;
// MLP layers are per-thread outer products: the layer input sits in a per-thread shared-memory column
// (conflict-free), weights are transposed [in][out] in shared memory and read as warp-broadcast float4,
// outputs accumulate in registers.  Persistent grid-stride over blocks of NT points.
#pragma once
#include "hr_device.cuh"

namespace hr {

// prepared weight block (floats), built on the host at create: transposed [in][out], padded
namespace wo_ {
constexpr int B_W1 = 0, B_b1 = 2048, B_W2 = 2112, B_b2 = 6208, B_W3 = 6272, B_b3 = 6784, B_SIZE = 6792;
constexpr int I_W1f = 0, I_W1w = 2048, I_b1 = 2304, I_W2 = 2368, I_b2 = 6464, I_W3 = 6528, I_b3 = 6656, I_SIZE = 6660;
constexpr int ALL = B_SIZE + I_SIZE;
}  // namespace wo_

constexpr int kMaxS2 = 64;   // tertiary directions (shared set) staged per block

template <int K, int J, int NT>
__device__ __forceinline__ void dense_acc(const float* __restrict__ Wt, const float* __restrict__ scr, float (&acc)[J]) {
#pragma unroll 4
  for (int k = 0; k < K; ++k) {
    const float a = scr[k * NT];
    const float4* w = reinterpret_cast<const float4*>(Wt + k * J);
#pragma unroll
    for (int j = 0; j < J / 4; ++j) {
      const float4 ww = w[j];
      acc[4 * j + 0] = fmaf(a, ww.x, acc[4 * j + 0]);
      acc[4 * j + 1] = fmaf(a, ww.y, acc[4 * j + 1]);
      acc[4 * j + 2] = fmaf(a, ww.z, acc[4 * j + 2]);
      acc[4 * j + 3] = fmaf(a, ww.w, acc[4 * j + 3]);
    }
  }
}

template <int J>
__device__ __forceinline__ void load_bias(const float* __restrict__ b, float (&acc)[J]) {
#pragma unroll
  for (int j = 0; j < J / 4; ++j) {
    const float4 v = reinterpret_cast<const float4*>(b)[j];
    acc[4 * j] = v.x; acc[4 * j + 1] = v.y; acc[4 * j + 2] = v.z; acc[4 * j + 3] = v.w;
  }
}

// B(f): f already in scr[0..31]; returns post-activation brdf.  Clobbers scr[0..63].
template <int NT>
__device__ __forceinline__ void brdf_decode_scr(const ShadeP& sp, const float* __restrict__ wB, float* scr, float (&brdf)[7]) {
  float h[kH];
  load_bias<kH>(wB + wo_::B_b1, h);
  dense_acc<kD, kH, NT>(wB + wo_::B_W1, scr, h);
#pragma unroll
  for (int k = 0; k < kH; ++k) scr[k * NT] = fmaxf(h[k], 0.f);
  load_bias<kH>(wB + wo_::B_b2, h);
  dense_acc<kH, kH, NT>(wB + wo_::B_W2, scr, h);
  float o[8];
  load_bias<8>(wB + wo_::B_b3, o);
#pragma unroll
  for (int k = 0; k < kH; ++k) {
    const float a = fmaxf(h[k], 0.f);
    const float4 w0 = reinterpret_cast<const float4*>(wB + wo_::B_W3 + k * 8)[0];
    const float4 w1 = reinterpret_cast<const float4*>(wB + wo_::B_W3 + k * 8)[1];
    o[0] = fmaf(a, w0.x, o[0]); o[1] = fmaf(a, w0.y, o[1]); o[2] = fmaf(a, w0.z, o[2]); o[3] = fmaf(a, w0.w, o[3]);
    o[4] = fmaf(a, w1.x, o[4]); o[5] = fmaf(a, w1.y, o[5]); o[6] = fmaf(a, w1.z, o[6]);
  }
  brdf_maps(sp, o, brdf);
}

// Layers 2+3 of I with h1 already in scr[0..63] -> raw (z_v, z_t).
template <int NT>
__device__ __forceinline__ void irt_tail_scr(const float* __restrict__ wI, const float* scr, float& zv, float& zt) {
  float h[kH];
  load_bias<kH>(wI + wo_::I_b2, h);
  dense_acc<kH, kH, NT>(wI + wo_::I_W2, scr, h);
  zv = wI[wo_::I_b3]; zt = wI[wo_::I_b3 + 1];
#pragma unroll
  for (int k = 0; k < kH; ++k) {
    const float a = fmaxf(h[k], 0.f);
    const float2 w = reinterpret_cast<const float2*>(wI + wo_::I_W3)[k];
    zv = fmaf(a, w.x, zv); zt = fmaf(a, w.y, zt);
  }
}

// h1 = relu(P + W1w . w) into scr, P read through `Pk(k)`.
template <int NT, typename PF>
__device__ __forceinline__ void irt_h1_to_scr(const float* __restrict__ wI, float* scr, PF Pk, float wx, float wy, float wz) {
#pragma unroll
  for (int k = 0; k < kH; ++k) {
    float a = fmaf(wI[wo_::I_W1w + k], wx, Pk(k));
    a = fmaf(wI[wo_::I_W1w + kH + k], wy, a);
    a = fmaf(wI[wo_::I_W1w + 2 * kH + k], wz, a);
    scr[k * NT] = fmaxf(a, 0.f);
  }
}

constexpr size_t ffma_smem_bytes(int NT, bool with_P) {
  return (size_t)(wo_::ALL + NT * kH * (with_P ? 2 : 1) + kMaxS2 * (kH + 3)) * sizeof(float);
}

__device__ __forceinline__ void load_weights_smem(float* sw, const float* __restrict__ wts, int nthreads) {
  const float4* src = reinterpret_cast<const float4*>(wts);
  float4* dst = reinterpret_cast<float4*>(sw);
  for (int i = threadIdx.x; i < wo_::ALL / 4; i += nthreads) dst[i] = __ldg(src + i);
}

// ---------------------------------------------------------------------------------------------------------
// encode: one thread per point (a1-a4)
template <bool F16>
__global__ void __launch_bounds__(256) k_encode(GridP g, const float* __restrict__ x, unsigned long long N,
                                                float* __restrict__ feat, uint32_t* __restrict__ idx, float* __restrict__ w) {
  const uint32_t D = g.L * 2;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < N;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    const float px = __ldg(x + 3 * i), py = __ldg(x + 3 * i + 1), pz = __ldg(x + 3 * i + 2);
    for (int l = 0; l < (int)g.L; ++l) {
      uint32_t id[8]; float ww[3];
      const float2 v = encode_level<F16>(g, l, px, py, pz, id, ww);
      feat[i * D + 2 * l] = v.x; feat[i * D + 2 * l + 1] = v.y;
      if (idx) {
#pragma unroll
        for (int k = 0; k < 8; ++k) idx[(i * g.L + l) * 8 + k] = id[k];
      }
      if (w) { w[(i * g.L + l) * 3] = ww[0]; w[(i * g.L + l) * 3 + 1] = ww[1]; w[(i * g.L + l) * 3 + 2] = ww[2]; }
    }
  }
}

// decode: B(f) per point (a5)
template <int NT>
__global__ void __launch_bounds__(NT, 1) k_decode_ffma(ShadeP sp, const float* __restrict__ wts, uint32_t D,
                                                       const float* __restrict__ feat, unsigned long long N, float* __restrict__ brdf) {
  extern __shared__ float4 smem4[];
  float* sw = reinterpret_cast<float*>(smem4);
  float* scr = sw + wo_::ALL + threadIdx.x;
  load_weights_smem(sw, wts, NT);
  __syncthreads();
  const float* wB = sw;
  for (unsigned long long i = blockIdx.x * (unsigned long long)NT + threadIdx.x; i < N; i += (unsigned long long)gridDim.x * NT) {
#pragma unroll
    for (int k = 0; k < kD; ++k) scr[k * NT] = (k < (int)D) ? __ldg(feat + i * D + k) : 0.f;
    float b[7];
    brdf_decode_scr<NT>(sp, wB, scr, b);
#pragma unroll
    for (int k = 0; k < 7; ++k) brdf[i * 7 + k] = b[k];
  }
}

// trace: I(f, w) for all directions of a set (+ fused encode when feat == NULL), x' (a6, a7)
template <bool F16, int NT>
__global__ void __launch_bounds__(NT, 1) k_trace_ffma(GridP g, ShadeP sp, const float* __restrict__ wts, const float* __restrict__ x,
                                                      const float* __restrict__ feat, unsigned long long N, DirsetP ds,
                                                      float* __restrict__ vis, float* __restrict__ zvo, float* __restrict__ to,
                                                      float* __restrict__ xsec) {
  extern __shared__ float4 smem4[];
  float* sw = reinterpret_cast<float*>(smem4);
  float* scr = sw + wo_::ALL + threadIdx.x;
  load_weights_smem(sw, wts, NT);
  __syncthreads();
  const float* wI = sw + wo_::B_SIZE;
  const uint32_t D = g.L * 2;
  for (unsigned long long i = blockIdx.x * (unsigned long long)NT + threadIdx.x; i < N; i += (unsigned long long)gridDim.x * NT) {
    float px = 0.f, py = 0.f, pz = 0.f;
    if (x) { px = __ldg(x + 3 * i); py = __ldg(x + 3 * i + 1); pz = __ldg(x + 3 * i + 2); }
    if (feat) {
#pragma unroll
      for (int k = 0; k < kD; ++k) scr[k * NT] = (k < (int)D) ? __ldg(feat + i * D + k) : 0.f;
    } else {
      float f[kD];
      encode_point<F16>(g, px, py, pz, f);
#pragma unroll
      for (int k = 0; k < kD; ++k) scr[k * NT] = f[k];
    }
    float P[kH];
    load_bias<kH>(wI + wo_::I_b1, P);
    dense_acc<kD, kH, NT>(wI + wo_::I_W1f, scr, P);
    for (uint32_t s = 0; s < ds.S; ++s) {
      const float* dp = dir_of(ds, i, s);
      const float wx = __ldg(dp), wy = __ldg(dp + 1), wz = __ldg(dp + 2);
      irt_h1_to_scr<NT>(wI, scr, [&](int k) { return P[k]; }, wx, wy, wz);
      float zv, zt, v, t;
      irt_tail_scr<NT>(wI, scr, zv, zt);
      irt_maps(sp, zv, zt, v, t);
      const unsigned long long o = i * ds.S + s;
      vis[o] = v; to[o] = t;
      if (zvo) zvo[o] = zv;
      if (xsec) { xsec[o * 3] = sec_hit(px, t, wx); xsec[o * 3 + 1] = sec_hit(py, t, wy); xsec[o * 3 + 2] = sec_hit(pz, t, wz); }
    }
  }
}

// shade: Eq. 1 with Eq. 2 per direction on one set (a9-a11)
static __global__ void __launch_bounds__(256) k_shade(EnvP env, ShadeP sp, const float* __restrict__ brdf, const float* __restrict__ wo,
                                               unsigned long long N, DirsetP ds, const float* __restrict__ vis,
                                               const float* __restrict__ Lind, uint32_t terms, float* __restrict__ rgb) {
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < N;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    float b[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) b[k] = __ldg(brdf + i * 7 + k);
    const float ox = __ldg(wo + 3 * i), oy = __ldg(wo + 3 * i + 1), oz = __ldg(wo + 3 * i + 2);
    float r = 0.f, gch = 0.f, bch = 0.f;
    for (uint32_t s = 0; s < ds.S; ++s) {
      const float* dp = dir_of(ds, i, s);
      const float wx = __ldg(dp), wy = __ldg(dp + 1), wz = __ldg(dp + 2);
      const float3 g = brdf_cos_over_pdf(sp, b, wx, wy, wz, ox, oy, oz, pdf_of(ds, i, s));
      const float v = __ldg(vis + i * ds.S + s);
      float3 L = make_float3(0.f, 0.f, 0.f);
      if (terms & 1u) { const float3 e = incoming(env, ds, i, s, wx, wy, wz); L = make_float3(v * e.x, v * e.y, v * e.z); }
      if ((terms & 2u) && Lind) {
        const float* lp = Lind + (i * ds.S + s) * 3;
        L.x += (1.f - v) * __ldg(lp); L.y += (1.f - v) * __ldg(lp + 1); L.z += (1.f - v) * __ldg(lp + 2);
      }
      r = fmaf(L.x, g.x, r); gch = fmaf(L.y, g.y, gch); bch = fmaf(L.z, g.z, bch);
    }
    const float inv = 1.f / (float)ds.S;
    rgb[3 * i] = r * inv; rgb[3 * i + 1] = gch * inv; rgb[3 * i + 2] = bch * inv;
  }
}

// L'_o at a secondary point (a8): f' = H(x'), B(f'), I(f', w'_k) over the tertiary set, Eq. 1 with w_o' = -w_j.
template <bool F16, int NT>
__device__ __forceinline__ float3 secondary_radiance_ffma(const GridP& g, const EnvP& env, const ShadeP& sp, const float* __restrict__ wB,
                                                          const float* __restrict__ wI, float* scr, float xs, float ys, float zs,
                                                          float ox, float oy, float oz, const DirsetP& tt, unsigned long long trow,
                                                          const float* __restrict__ Qt, const float* __restrict__ Lt) {
  {
    float f[kD];
    encode_point<F16>(g, xs, ys, zs, f);
#pragma unroll
    for (int k = 0; k < kD; ++k) scr[k * NT] = f[k];
  }
  float P2[kH];
  load_bias<kH>(wI + wo_::I_b1, P2);
  dense_acc<kD, kH, NT>(wI + wo_::I_W1f, scr, P2);
  float b[7];
  brdf_decode_scr<NT>(sp, wB, scr, b);
  float r = 0.f, gch = 0.f, bch = 0.f;
  const bool shared = tt.stride == 0;
  for (uint32_t k = 0; k < tt.S; ++k) {
    const float* dp = dir_of(tt, trow, k);
    const float wx = __ldg(dp), wy = __ldg(dp + 1), wz = __ldg(dp + 2);
    if (shared) {
#pragma unroll
      for (int q = 0; q < kH; ++q) scr[q * NT] = fmaxf(P2[q] + Qt[k * kH + q], 0.f);
    } else {
      irt_h1_to_scr<NT>(wI, scr, [&](int q) { return P2[q]; }, wx, wy, wz);
    }
    float zv, zt, v, t;
    irt_tail_scr<NT>(wI, scr, zv, zt);
    irt_maps(sp, zv, zt, v, t);
    const float3 gg = brdf_cos_over_pdf(sp, b, wx, wy, wz, ox, oy, oz, pdf_of(tt, trow, k));
    float3 L;
    if (shared && !tt.Lin) L = make_float3(Lt[k * 3], Lt[k * 3 + 1], Lt[k * 3 + 2]);
    else L = incoming(env, tt, trow, k, wx, wy, wz);
    r = fmaf(v * L.x, gg.x, r); gch = fmaf(v * L.y, gg.y, gch); bch = fmaf(v * L.z, gg.z, bch);
  }
  const float inv = 1.f / (float)tt.S;
  return make_float3(r * inv, gch * inv, bch * inv);
}

// render_frame: all of a1-a11 fused, one thread per primary point.
template <bool F16, int NT>
__global__ void __launch_bounds__(NT, 1) k_render_ffma(GridP g, EnvP env, ShadeP sp, const float* __restrict__ wts, FrameP fr,
                                                       float* __restrict__ rgb) {
  extern __shared__ float4 smem4[];
  float* sw = reinterpret_cast<float*>(smem4);
  float* scr = sw + wo_::ALL + threadIdx.x;
  float* Ps = sw + wo_::ALL + NT * kH + threadIdx.x;
  float* Qt = sw + wo_::ALL + 2 * NT * kH;        // [S2][64] = W1w . w'_k for the shared tertiary set
  float* Lt = Qt + kMaxS2 * kH;                   // [S2][3] radiance of the shared tertiary set
  load_weights_smem(sw, wts, NT);
  __syncthreads();
  const float* wB = sw;
  const float* wI = sw + wo_::B_SIZE;
  const bool indirect = (fr.flags & 4u) && fr.s.S && fr.t.S;
  if (indirect && fr.t.stride == 0) {
    for (int e = threadIdx.x; e < (int)fr.t.S * kH; e += NT) {
      const int k = e / kH, q = e % kH;
      const float* dp = fr.t.dir + 3 * k;
      Qt[e] = wI[wo_::I_W1w + q] * __ldg(dp) + wI[wo_::I_W1w + kH + q] * __ldg(dp + 1) + wI[wo_::I_W1w + 2 * kH + q] * __ldg(dp + 2);
    }
    if (!fr.t.Lin)
      for (int k = threadIdx.x; k < (int)fr.t.S; k += NT) {
        const float* dp = fr.t.dir + 3 * k;
        const float3 L = env_lookup(env, __ldg(dp), __ldg(dp + 1), __ldg(dp + 2));
        Lt[3 * k] = L.x; Lt[3 * k + 1] = L.y; Lt[3 * k + 2] = L.z;
      }
  }
  __syncthreads();
  for (unsigned long long i = blockIdx.x * (unsigned long long)NT + threadIdx.x; i < fr.N; i += (unsigned long long)gridDim.x * NT) {
    if (fr.mask && !fr.mask[i]) { rgb[3 * i] = 0.f; rgb[3 * i + 1] = 0.f; rgb[3 * i + 2] = 0.f; continue; }
    const float px = __ldg(fr.x + 3 * i), py = __ldg(fr.x + 3 * i + 1), pz = __ldg(fr.x + 3 * i + 2);
    const float ox = __ldg(fr.wo + 3 * i), oy = __ldg(fr.wo + 3 * i + 1), oz = __ldg(fr.wo + 3 * i + 2);
    float b[7];
    {
      float f[kD];
      encode_point<F16>(g, px, py, pz, f);
#pragma unroll
      for (int k = 0; k < kD; ++k) scr[k * NT] = f[k];
      float P[kH];
      load_bias<kH>(wI + wo_::I_b1, P);
      dense_acc<kD, kH, NT>(wI + wo_::I_W1f, scr, P);
#pragma unroll
      for (int k = 0; k < kH; ++k) Ps[k * NT] = P[k];
      if (fr.brdf) {
#pragma unroll
        for (int k = 0; k < 7; ++k) b[k] = __ldg(fr.brdf + i * 7 + k);
      } else {
        brdf_decode_scr<NT>(sp, wB, scr, b);
      }
    }
    float r = 0.f, gch = 0.f, bch = 0.f;
    if ((fr.flags & 1u) && fr.d.S) {                                  // direct term of Eq. 1
      float ar = 0.f, ag = 0.f, ab = 0.f;
      for (uint32_t s = 0; s < fr.d.S; ++s) {
        const float* dp = dir_of(fr.d, i, s);
        const float wx = __ldg(dp), wy = __ldg(dp + 1), wz = __ldg(dp + 2);
        float v = 1.f;
        if (fr.flags & 2u) {
          irt_h1_to_scr<NT>(wI, scr, [&](int k) { return Ps[k * NT]; }, wx, wy, wz);
          float zv, zt, t;
          irt_tail_scr<NT>(wI, scr, zv, zt);
          irt_maps(sp, zv, zt, v, t);
        }
        const float3 gg = brdf_cos_over_pdf(sp, b, wx, wy, wz, ox, oy, oz, pdf_of(fr.d, i, s));
        const float3 L = incoming(env, fr.d, i, s, wx, wy, wz);
        ar = fmaf(v * L.x, gg.x, ar); ag = fmaf(v * L.y, gg.y, ag); ab = fmaf(v * L.z, gg.z, ab);
      }
      const float inv = 1.f / (float)fr.d.S;
      r = ar * inv; gch = ag * inv; bch = ab * inv;
    }
    if (indirect) {                                                   // (1 - V) L'_o term of Eq. 2
      float ar = 0.f, ag = 0.f, ab = 0.f;
      for (uint32_t j = 0; j < fr.s.S; ++j) {
        const float* dp = dir_of(fr.s, i, j);
        const float wx = __ldg(dp), wy = __ldg(dp + 1), wz = __ldg(dp + 2);
        irt_h1_to_scr<NT>(wI, scr, [&](int k) { return Ps[k * NT]; }, wx, wy, wz);
        float zv, zt, v, t;
        irt_tail_scr<NT>(wI, scr, zv, zt);
        irt_maps(sp, zv, zt, v, t);
        const float3 Lo = secondary_radiance_ffma<F16, NT>(g, env, sp, wB, wI, scr, sec_hit(px, t, wx), sec_hit(py, t, wy),
                                                           sec_hit(pz, t, wz), -wx, -wy, -wz, fr.t,
                                                           fr.t.stride ? i * fr.s.S + j : 0ull, Qt, Lt);
        const float3 gg = brdf_cos_over_pdf(sp, b, wx, wy, wz, ox, oy, oz, pdf_of(fr.s, i, j));
        const float m = 1.f - v;
        ar = fmaf(m * Lo.x, gg.x, ar); ag = fmaf(m * Lo.y, gg.y, ag); ab = fmaf(m * Lo.z, gg.z, ab);
      }
      const float inv = 1.f / (float)fr.s.S;
      r = fmaf(ar, inv, r); gch = fmaf(ag, inv, gch); bch = fmaf(ab, inv, bch);
    }
    rgb[3 * i] = r; rgb[3 * i + 1] = gch; rgb[3 * i + 2] = bch;
  }
}

}  // namespace hr
