// hr_sampler.cuh -- on-device direction sampler for the hash-grid renderer.
//   MIS of a light-importance ray and a GGX visible-normal ray per primary point and sample, every ray carrying the
//   balance-heuristic pdf (p_light + p_ggx) / 2; alpha = Roughness^2.   PAPER.md:344 / 338: stratified ray sets.
// Definitions are DESIGN.md readings Q35-Q38.  fp32 arithmetic; the discrete decisions (24-bit uniforms, the stratified CDF
// coordinate and its comparison against the fp32 CDF table) are single IEEE operations so they are bit-reproducible.
// The kernels only write direction / pdf arrays (16 bytes per ray): they are bound by the HBM store stream.
#pragma once
#include <stdint.h>

namespace hr {
namespace smp {

constexpr float kPiF = 3.14159265358979f;

// Q35: counter-based generator -- a 32-bit multiply-xorshift finalizer chained over (seed, row, sample, dimension)
__device__ __forceinline__ uint32_t mix32(uint32_t h) {
  h ^= h >> 16; h *= 0x7feb352du; h ^= h >> 15; h *= 0x846ca68bu; h ^= h >> 16;
  return h;
}
__device__ __forceinline__ uint32_t rng_prefix(unsigned long long seed, unsigned long long row) {
  uint32_t h = mix32((uint32_t)seed ^ 0x9E3779B9u);
  h = mix32(h ^ (uint32_t)(seed >> 32));
  h = mix32(h ^ (uint32_t)row);
  h = mix32(h ^ (uint32_t)(row >> 32));
  return h;
}
__device__ __forceinline__ float rng_uniform(uint32_t prefix, uint32_t sample, uint32_t dim) {
  const uint32_t r = mix32(mix32(prefix ^ (sample * 16u + dim)) + 0x9E3779B9u);
  return __uint2float_rz(r >> 8) * 5.9604644775390625e-8f;          // [0, 1), exact
}

// Q36: orthonormal frame of a unit normal (branchless construction of Duff et al. 2017)
__device__ __forceinline__ void frame_of(float nx, float ny, float nz, float3& T, float3& B) {
  const float sign = nz >= 0.f ? 1.f : -1.f;
  const float a = -1.f / (sign + nz);
  const float b = nx * ny * a;
  T = make_float3(1.f + sign * nx * nx * a, sign * b, -sign * nx);
  B = make_float3(b, sign + ny * ny * a, -ny);
}

struct LightP { const float* pmf; const float* cdf; uint32_t He, We; };

// Q37: density (w.r.t. solid angle) of the light-importance strategy at direction w
__device__ __forceinline__ float light_pdf(const LightP& lp, float wx, float wy, float wz) {
  const float theta = acosf(fminf(fmaxf(wz, -1.f), 1.f)), phi = atan2f(wy, wx);
  int r = (int)floorf(theta * (1.f / kPiF) * (float)lp.He); r = min(max(r, 0), (int)lp.He - 1);
  int c = (int)floorf((phi * (0.5f / kPiF) + 0.5f) * (float)lp.We); c = min(max(c, 0), (int)lp.We - 1);
  const float st = fmaxf(sinf(theta), 1e-9f);
  return __ldg(lp.pmf + r * lp.We + c) / ((kPiF / (float)lp.He) * (2.f * kPiF / (float)lp.We) * st);
}

// Q38: GGX visible-normal distribution (Heitz 2018), isotropic, local frame z = normal
__device__ __forceinline__ float ggx_pdf_local(float alpha, float3 V, float3 L) {
  float3 H = make_float3(V.x + L.x, V.y + L.y, V.z + L.z);
  const float hn = rsqrtf(fmaxf(H.x * H.x + H.y * H.y + H.z * H.z, 1e-30f));
  H.z *= hn;
  if (!(H.z > 0.f)) return 0.f;
  const float k = alpha * alpha;
  const float dd = k * H.z * H.z + (H.x * H.x + H.y * H.y) * hn * hn;      // = H.z^2 (k - 1) + 1 without the cancellation
  const float D = k / (kPiF * dd * dd);
  const float G1 = 2.f * V.z / (V.z + sqrtf(k + (1.f - k) * V.z * V.z));
  return G1 * D / (4.f * V.z);
}
__device__ __forceinline__ float3 ggx_sample_local(float alpha, float3 V, float u1, float u2) {
  float3 Vh = make_float3(alpha * V.x, alpha * V.y, V.z);
  const float vn = rsqrtf(Vh.x * Vh.x + Vh.y * Vh.y + Vh.z * Vh.z);
  Vh.x *= vn; Vh.y *= vn; Vh.z *= vn;
  float3 T1 = make_float3(1.f, 0.f, 0.f);
  const float lensq = Vh.x * Vh.x + Vh.y * Vh.y;
  if (lensq > 1e-14f) { const float inv = rsqrtf(lensq); T1 = make_float3(-Vh.y * inv, Vh.x * inv, 0.f); }
  const float3 T2 = make_float3(Vh.y * T1.z - Vh.z * T1.y, Vh.z * T1.x - Vh.x * T1.z, Vh.x * T1.y - Vh.y * T1.x);
  const float r = sqrtf(u1), phi = 2.f * kPiF * u2;
  float sp, cp;
  sincosf(phi, &sp, &cp);
  const float t1 = r * cp;
  float t2 = r * sp;
  const float s = 0.5f * (1.f + Vh.z);
  t2 = (1.f - s) * sqrtf(fmaxf(1.f - t1 * t1, 0.f)) + s * t2;
  const float t3 = sqrtf(fmaxf(1.f - t1 * t1 - t2 * t2, 0.f));
  const float3 Nh = make_float3(t1 * T1.x + t2 * T2.x + t3 * Vh.x, t1 * T1.y + t2 * T2.y + t3 * Vh.y, t1 * T1.z + t2 * T2.z + t3 * Vh.z);
  float3 Ne = make_float3(alpha * Nh.x, alpha * Nh.y, fmaxf(Nh.z, 0.f));
  const float nn = rsqrtf(fmaxf(Ne.x * Ne.x + Ne.y * Ne.y + Ne.z * Ne.z, 1e-30f));
  Ne.x *= nn; Ne.y *= nn; Ne.z *= nn;
  const float vd = V.x * Ne.x + V.y * Ne.y + V.z * Ne.z;
  return make_float3(2.f * vd * Ne.x - V.x, 2.f * vd * Ne.y - V.y, 2.f * vd * Ne.z - V.z);
}

// One thread per (point, sample): slot 2s = light ray, slot 2s+1 = GGX ray; both pdfs = (p_light + p_ggx) / 2.
__global__ void __launch_bounds__(256) k_sample_mis(LightP lp, const float* __restrict__ brdf, const float* __restrict__ wo, unsigned long long N,
                                                    uint32_t spp, unsigned long long seed, float* __restrict__ dir, float* __restrict__ pdf) {
  const unsigned long long total = N * spp;
  const float inv_spp = __frcp_rn((float)spp);
  const uint32_t ntex = lp.He * lp.We;
  for (unsigned long long e = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; e < total; e += (unsigned long long)gridDim.x * blockDim.x) {
    const unsigned long long i = e / spp;
    const uint32_t s = (uint32_t)(e - i * spp);
    const uint32_t pre = rng_prefix(seed, i);
    const float nx = __ldg(brdf + 7 * i), ny = __ldg(brdf + 7 * i + 1), nz = __ldg(brdf + 7 * i + 2), rough = __ldg(brdf + 7 * i + 6);
    const float ox = __ldg(wo + 3 * i), oy = __ldg(wo + 3 * i + 1), oz = __ldg(wo + 3 * i + 2);
    const float alpha = rough * rough;
    float3 T, B;
    frame_of(nx, ny, nz, T, B);
    float3 V = make_float3(ox * T.x + oy * T.y + oz * T.z, ox * B.x + oy * B.y + oz * B.z, fmaxf(ox * nx + oy * ny + oz * nz, 1e-4f));
    const float vn = rsqrtf(V.x * V.x + V.y * V.y + V.z * V.z);
    V.x *= vn; V.y *= vn; V.z *= vn;
    // light ray: stratified CDF inversion (first k with cdf[k] > u0), jittered inside the texel
    const float u0 = __fmul_rn(__fadd_rn((float)s, rng_uniform(pre, s, 0)), inv_spp);
    uint32_t lo = 0, hi = ntex - 1;
    while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (__ldg(lp.cdf + mid) > u0) hi = mid; else lo = mid + 1; }
    const uint32_t r = lo / lp.We, c = lo - r * lp.We;
    const float theta = kPiF * ((float)r + rng_uniform(pre, s, 1)) / (float)lp.He;
    const float phi = 2.f * kPiF * ((float)c + rng_uniform(pre, s, 2)) / (float)lp.We - kPiF;
    float st, ct, sp, cp;
    sincosf(theta, &st, &ct);
    sincosf(phi, &sp, &cp);
    const float3 dl = make_float3(st * cp, st * sp, ct);
    // GGX visible-normal ray
    const float3 Lg = ggx_sample_local(alpha, V, rng_uniform(pre, s, 3), rng_uniform(pre, s, 4));
    const float3 dg = make_float3(Lg.x * T.x + Lg.y * B.x + Lg.z * nx, Lg.x * T.y + Lg.y * B.y + Lg.z * ny, Lg.x * T.z + Lg.y * B.z + Lg.z * nz);
    const float3 Ll = make_float3(dl.x * T.x + dl.y * T.y + dl.z * T.z, dl.x * B.x + dl.y * B.y + dl.z * B.z, dl.x * nx + dl.y * ny + dl.z * nz);
    const float pl = 0.5f * (light_pdf(lp, dl.x, dl.y, dl.z) + ggx_pdf_local(alpha, V, Ll));
    const float pg = 0.5f * (light_pdf(lp, dg.x, dg.y, dg.z) + ggx_pdf_local(alpha, V, Lg));
    float* d = dir + e * 6;
    d[0] = dl.x; d[1] = dl.y; d[2] = dl.z; d[3] = dg.x; d[4] = dg.y; d[5] = dg.z;
    reinterpret_cast<float2*>(pdf)[e] = make_float2(pl, pg);
  }
}

// One thread per (row, stratum): Sa x Sb jittered strata; normal != NULL: cosine hemisphere about normal[row] (pdf cos/pi),
// else whole sphere (pdf 1/4pi).  Stratum (a, b) -> slot a * Sb + b.
__global__ void __launch_bounds__(256) k_sample_stratified(const float* __restrict__ normal, unsigned long long rows, uint32_t Sa, uint32_t Sb,
                                                           unsigned long long seed, float* __restrict__ dir, float* __restrict__ pdf) {
  const uint32_t S = Sa * Sb;
  const unsigned long long total = rows * S;
  for (unsigned long long e = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; e < total; e += (unsigned long long)gridDim.x * blockDim.x) {
    const unsigned long long i = e / S;
    const uint32_t s = (uint32_t)(e - i * S), a = s / Sb, b = s - a * Sb;
    const uint32_t pre = rng_prefix(seed, i);
    const float u = ((float)a + rng_uniform(pre, s, 0)) / (float)Sa;
    const float v = ((float)b + rng_uniform(pre, s, 1)) / (float)Sb;
    float sp, cp;
    sincosf(2.f * kPiF * v, &sp, &cp);
    float3 d; float p;
    if (normal) {
      const float nx = __ldg(normal + 3 * i), ny = __ldg(normal + 3 * i + 1), nz = __ldg(normal + 3 * i + 2);
      float3 T, B;
      frame_of(nx, ny, nz, T, B);
      const float r = sqrtf(u), z = sqrtf(1.f - u);
      const float lx = r * cp, ly = r * sp;
      d = make_float3(lx * T.x + ly * B.x + z * nx, lx * T.y + ly * B.y + z * ny, lx * T.z + ly * B.z + z * nz);
      p = z * (1.f / kPiF);
    } else {
      const float z = 1.f - 2.f * u, r = sqrtf(fmaxf(1.f - z * z, 0.f));
      d = make_float3(r * cp, r * sp, z);
      p = 0.25f / kPiF;
    }
    dir[e * 3] = d.x; dir[e * 3 + 1] = d.y; dir[e * 3 + 2] = d.z;
    pdf[e] = p;
  }
}

}  // namespace smp
}  // namespace hr
