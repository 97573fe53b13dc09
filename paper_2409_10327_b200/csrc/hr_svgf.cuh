// hr_svgf.cuh -- spatial-only SVGF denoiser, the step after the hash-grid renderer.
//   "SVGF ... operates on the raw MC rendering results ... all temporal elements of SVGF are removed";
//   the depth gradient is the finite difference of the depth derived from the primary surface coordinate map.
// The filter is the published spatial part of SVGF (Schied et al. 2017), readings Q39-Q44 of DESIGN.md: albedo demodulation,
// 7x7 bilateral estimate of the luminance variance, `iterations` 5x5 a-trous passes with hole size 2^i, B3-spline kernel,
// edge-stopping weights w_z (depth, scaled by the gradient), w_n (normal, power sigma_n) and w_l (luminance, scaled by the
// 3x3-gaussian-filtered standard deviation), variance filtered with squared weights.
// One thread per pixel, every pass a stencil over L2-resident images (an 800x800 frame is 10 MB per float4 plane): bound by
// L2 / HBM bandwidth, 25 taps x 44 bytes per pixel and pass.  Depth is kept in fp64 so that |z_p - z_q|, a difference of
// nearly equal distances, does not lose the digits the depth weight needs.
#pragma once
#include <stdint.h>

namespace hr {
namespace svgf {

struct Geo { double z; float gx, gy; };       // depth, forward-difference gradient (backward on the last column / row)

struct Params {
  uint32_t H, W;
  float sigma_z, sigma_n, sigma_l;
  float cam[3];
};

__device__ __forceinline__ float luma(float4 c) { return 0.2126f * c.x + 0.7152f * c.y + 0.0722f * c.z; }

__device__ __forceinline__ double depth_at(const float* __restrict__ pos, const Params& P, uint32_t y, uint32_t x) {
  const float* p = pos + ((size_t)y * P.W + x) * 3;
  const double dx = (double)__ldg(p) - (double)P.cam[0], dy = (double)__ldg(p + 1) - (double)P.cam[1], dz = (double)__ldg(p + 2) - (double)P.cam[2];
  return sqrt(dx * dx + dy * dy + dz * dz);
}

// pass 0: depth + gradient, live flag, demodulated colour (variance slot zeroed)
__global__ void __launch_bounds__(256) k_svgf_prep(Params P, const float* __restrict__ rgb, const float* __restrict__ albedo,
                                                   const float* __restrict__ pos, const uint8_t* __restrict__ mask, Geo* __restrict__ geo,
                                                   uint8_t* __restrict__ live, float4* __restrict__ col) {
  const size_t n = (size_t)P.H * P.W;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const uint32_t y = (uint32_t)(i / P.W), x = (uint32_t)(i - (size_t)y * P.W);
    const double z = depth_at(pos, P, y, x);
    Geo g; g.z = z;
    if (P.W > 1) g.gx = x + 1 < P.W ? (float)(depth_at(pos, P, y, x + 1) - z) : (float)(z - depth_at(pos, P, y, x - 1)); else g.gx = 0.f;
    if (P.H > 1) g.gy = y + 1 < P.H ? (float)(depth_at(pos, P, y + 1, x) - z) : (float)(z - depth_at(pos, P, y - 1, x)); else g.gy = 0.f;
    geo[i] = g;
    live[i] = mask ? (mask[i] ? 1 : 0) : 1;
    float r = __ldg(rgb + 3 * i), gch = __ldg(rgb + 3 * i + 1), b = __ldg(rgb + 3 * i + 2);
    if (albedo) {
      r /= fmaxf(__ldg(albedo + 3 * i), 1e-3f); gch /= fmaxf(__ldg(albedo + 3 * i + 1), 1e-3f); b /= fmaxf(__ldg(albedo + 3 * i + 2), 1e-3f);
    }
    col[i] = make_float4(r, gch, b, 0.f);
  }
}

// w_z * w_n of the tap q = p + (dy, dx) (SVGF eq. 3, 4); the caller has checked that q is inside the image
__device__ __forceinline__ float geometry_weight(const Params& P, const Geo& gp, float3 np_, const Geo* __restrict__ geo,
                                                 const float* __restrict__ nrm, const uint8_t* __restrict__ live, size_t q, int dy, int dx) {
  if (!live[q]) return 0.f;
  const float adz = (float)fabs(gp.z - geo[q].z);
  const float wz = expf(-adz / (P.sigma_z * fabsf(gp.gx * (float)dx + gp.gy * (float)dy) + 1e-6f));
  const float d = fmaxf(np_.x * __ldg(nrm + 3 * q) + np_.y * __ldg(nrm + 3 * q + 1) + np_.z * __ldg(nrm + 3 * q + 2), 0.f);
  return wz * powf(d, P.sigma_n);
}

// pass 1: bilateral 7x7 first / second moments of the luminance -> variance (col.w)
__global__ void __launch_bounds__(256) k_svgf_variance(Params P, const Geo* __restrict__ geo, const float* __restrict__ nrm,
                                                       const uint8_t* __restrict__ live, float4* __restrict__ col) {
  const size_t n = (size_t)P.H * P.W;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    if (!live[i]) continue;
    const int y = (int)(i / P.W), x = (int)(i - (size_t)y * P.W);
    const Geo gp = geo[i];
    const float3 np_ = make_float3(__ldg(nrm + 3 * i), __ldg(nrm + 3 * i + 1), __ldg(nrm + 3 * i + 2));
    float s0 = 0.f, s1 = 0.f, s2 = 0.f;
    for (int dy = -3; dy <= 3; ++dy) {
      const int yy = y + dy;
      if (yy < 0 || yy >= (int)P.H) continue;
      for (int dx = -3; dx <= 3; ++dx) {
        const int xx = x + dx;
        if (xx < 0 || xx >= (int)P.W) continue;
        const size_t q = (size_t)yy * P.W + xx;
        const float w = geometry_weight(P, gp, np_, geo, nrm, live, q, dy, dx);
        const float* cq = reinterpret_cast<const float*>(col + q);          // rgb only: the .w slots are being written in this pass
        const float l = 0.2126f * cq[0] + 0.7152f * cq[1] + 0.0722f * cq[2];
        s0 += w; s1 += w * l; s2 += w * l * l;
      }
    }
    s0 = fmaxf(s0, 1e-12f);
    const float m1 = s1 / s0, m2 = s2 / s0;
    // the .w slot of OTHER pixels is not read in this pass, so writing ours in place is race-free
    col[i].w = fmaxf(0.f, m2 - m1 * m1);
  }
}

// pass 2..: one 5x5 a-trous iteration with hole size `step` (SVGF eq. 1, 2, 5).  last: remodulate, mask and write rgb.
__global__ void __launch_bounds__(256) k_svgf_atrous(Params P, int step, const Geo* __restrict__ geo, const float* __restrict__ nrm,
                                                     const uint8_t* __restrict__ live, const float4* __restrict__ in, float4* __restrict__ out,
                                                     const float* __restrict__ albedo, float* __restrict__ rgb_out) {
  const float h[5] = {1.f / 16.f, 1.f / 4.f, 3.f / 8.f, 1.f / 4.f, 1.f / 16.f};
  const size_t n = (size_t)P.H * P.W;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int y = (int)(i / P.W), x = (int)(i - (size_t)y * P.W);
    float4 res = in[i];
    if (live[i]) {
      const Geo gp = geo[i];
      const float3 np_ = make_float3(__ldg(nrm + 3 * i), __ldg(nrm + 3 * i + 1), __ldg(nrm + 3 * i + 2));
      const float lp = luma(res);
      float gv = 0.f, gw = 0.f;                       // 3x3 gaussian prefilter of the variance
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          const int yy = y + dy, xx = x + dx;
          if (yy < 0 || yy >= (int)P.H || xx < 0 || xx >= (int)P.W) continue;
          const float k = (dy ? 1.f : 2.f) * (dx ? 1.f : 2.f) * (1.f / 16.f);
          gv += k * in[(size_t)yy * P.W + xx].w; gw += k;
        }
      const float sd = sqrtf(fmaxf(gv / fmaxf(gw, 1e-12f), 0.f));
      const float inv_l = 1.f / (P.sigma_l * sd + 1e-6f);
      float nr = 0.f, ng = 0.f, nb = 0.f, den = 0.f, vn = 0.f;
      for (int iy = 0; iy < 5; ++iy) {
        const int dy = (iy - 2) * step, yy = y + dy;
        if (yy < 0 || yy >= (int)P.H) continue;
        for (int ix = 0; ix < 5; ++ix) {
          const int dx = (ix - 2) * step, xx = x + dx;
          if (xx < 0 || xx >= (int)P.W) continue;
          const size_t q = (size_t)yy * P.W + xx;
          float w = geometry_weight(P, gp, np_, geo, nrm, live, q, dy, dx);
          const float4 cq = in[q];
          w *= h[iy] * h[ix] * expf(-fabsf(lp - luma(cq)) * inv_l);
          nr += w * cq.x; ng += w * cq.y; nb += w * cq.z; den += w; vn += w * w * cq.w;
        }
      }
      if (den > 0.f) {
        const float inv = 1.f / fmaxf(den, 1e-12f);
        res = make_float4(nr * inv, ng * inv, nb * inv, vn * inv * inv);
      }
    }
    if (out) out[i] = res;
    if (rgb_out) {
      float r = res.x, g = res.y, b = res.z;
      if (albedo) { r *= fmaxf(__ldg(albedo + 3 * i), 1e-3f); g *= fmaxf(__ldg(albedo + 3 * i + 1), 1e-3f); b *= fmaxf(__ldg(albedo + 3 * i + 2), 1e-3f); }
      const bool on = live[i];
      rgb_out[3 * i] = on ? r : 0.f; rgb_out[3 * i + 1] = on ? g : 0.f; rgb_out[3 * i + 2] = on ? b : 0.f;
    }
  }
}

}  // namespace svgf
}  // namespace hr
