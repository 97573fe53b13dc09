// oracle/sampler_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain CPU statement of the direction sampler that feeds the hash-grid renderer:
//   * PAPER.md:122 (section 4.1): "we apply MIS where a light importance ray and a GGX importance ray are sampled for
//     each primary surface point.  The probability distribution function for the rays is computed with Veach's balance
//     heuristic.  The GGX rays are drawn from visible normal distribution function [8]"; alpha = Roughness^2, k = alpha^2.
//   * "we cast 8 random rays from each secondary surface point via stratified sampling"; PAPER.md:338:
//     stratified sampling on the whole sphere.
// Double precision throughout, EXCEPT the discrete decisions, which are defined in fp32 so that both sides take them
// identically (readings Q35-Q38): the uniform variate u = (r >> 8) * 2^-24 (exact), the stratified CDF
// coordinate u0 = fl32(fl32(s + xi) * fl32(1 / spp)) and the comparison against the fp32 CDF table.
// Shares no code with paper_2409_10327_b200/ and never includes include/hashrender.h.
//
// Pins (tests/test_sampler_pins.py): uniformity / independence of the counter-based generator, the light pmf summing to
// one and reproducing a one-hot map, the texel pdf integrating to one over the sphere, the VNDF pdf integrating to one
// (quadrature) and matching the empirical histogram of its own samples, exact one-sample-per-stratum occupancy, the
// balance-heuristic estimator reproducing closed-form integrals (constant env, Lambert: a*L).
#include <cmath>
#include <cstdint>
#include <vector>

namespace {

const double kPi = 3.14159265358979323846;

// ---- Q35: counter-based generator -------------------------------------------------------------------------------------
// A 32-bit multiply-xorshift finalizer (two multiplies, three xor-shifts), chained over (seed, row, sample, dimension).
inline uint32_t mix32(uint32_t h) {
  h ^= h >> 16; h *= 0x7feb352du; h ^= h >> 15; h *= 0x846ca68bu; h ^= h >> 16;
  return h;
}
inline uint32_t rng_prefix(uint64_t seed, uint64_t row) {
  uint32_t h = mix32((uint32_t)seed ^ 0x9E3779B9u);
  h = mix32(h ^ (uint32_t)(seed >> 32));
  h = mix32(h ^ (uint32_t)row);
  h = mix32(h ^ (uint32_t)(row >> 32));
  return h;
}
inline uint32_t rng_bits(uint32_t prefix, uint32_t sample, uint32_t dim) {
  return mix32(mix32(prefix ^ (sample * 16u + dim)) + 0x9E3779B9u);
}
inline float rng_uniform(uint32_t prefix, uint32_t sample, uint32_t dim) {      // [0, 1), exact in fp32
  return (float)(rng_bits(prefix, sample, dim) >> 8) * 5.9604644775390625e-8f;
}

inline void normalize3(double v[3]) {
  const double n = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
  const double inv = 1.0 / (n > 1e-300 ? n : 1e-300);
  v[0] *= inv; v[1] *= inv; v[2] *= inv;
}

// ---- Q36: orthonormal frame (T, B, n) of a unit normal: the branchless construction of Duff et al. 2017 ------------------
inline void frame_of(const double n[3], double T[3], double B[3]) {
  const double sign = n[2] >= 0.0 ? 1.0 : -1.0;
  const double a = -1.0 / (sign + n[2]);
  const double b = n[0] * n[1] * a;
  T[0] = 1.0 + sign * n[0] * n[0] * a; T[1] = sign * b; T[2] = -sign * n[0];
  B[0] = b; B[1] = sign + n[1] * n[1] * a; B[2] = -n[1];
}

// ---- Q37: light importance sampling of the equirect env map -----------------------------------------
// pmf over texels proportional to luminance * sin(theta of the row centre); the direction is uniform in (theta, phi) inside
// the chosen texel; density w.r.t. solid angle = pmf / (dtheta * dphi * sin theta).  Same (theta, phi) convention as the
// env lookup: theta from +z, phi = atan2(y, x), column c covers phi in [2 pi c / We - pi, 2 pi (c+1) / We - pi).
void build_light_tables(const float* env, uint32_t He, uint32_t We, std::vector<double>& pmf, std::vector<float>& cdf) {
  const size_t n = (size_t)He * We;
  pmf.assign(n, 0.0); cdf.assign(n, 0.f);
  double tot = 0.0;
  for (uint32_t r = 0; r < He; ++r) {
    const double st = std::sin(kPi * (r + 0.5) / He);
    for (uint32_t c = 0; c < We; ++c) {
      const float* p = env + ((size_t)r * We + c) * 3;
      const double Y = 0.2126 * (double)p[0] + 0.7152 * (double)p[1] + 0.0722 * (double)p[2];
      pmf[(size_t)r * We + c] = (Y > 0.0 ? Y : 0.0) * st;
      tot += pmf[(size_t)r * We + c];
    }
  }
  if (!(tot > 0.0)) {                           // black map: fall back to uniform-in-solid-angle rows
    tot = 0.0;
    for (uint32_t r = 0; r < He; ++r)
      for (uint32_t c = 0; c < We; ++c) { pmf[(size_t)r * We + c] = std::sin(kPi * (r + 0.5) / He); tot += pmf[(size_t)r * We + c]; }
  }
  double run = 0.0;
  for (size_t k = 0; k < n; ++k) { pmf[k] /= tot; run += pmf[k]; cdf[k] = (float)run; }
  cdf[n - 1] = 1.0f;
}
inline double light_pdf(const std::vector<double>& pmf, uint32_t He, uint32_t We, const double w[3]) {
  const double ct = w[2] < -1.0 ? -1.0 : (w[2] > 1.0 ? 1.0 : w[2]);
  const double theta = std::acos(ct), phi = std::atan2(w[1], w[0]);
  int r = (int)std::floor(theta / kPi * He); r = r < 0 ? 0 : (r >= (int)He ? (int)He - 1 : r);
  int c = (int)std::floor((phi / (2.0 * kPi) + 0.5) * We); c = c < 0 ? 0 : (c >= (int)We ? (int)We - 1 : c);
  const double st = std::sin(theta);
  return pmf[(size_t)r * We + c] / ((kPi / He) * (2.0 * kPi / We) * (st > 1e-9 ? st : 1e-9));
}

// ---- Q38: GGX visible-normal sampling (Heitz 2018), isotropic, alpha = r^2 ------------------------------
// V is the view direction in the local frame (z = normal); a view at or below the horizon is lifted to z = 1e-4.
inline void local_view(const double n[3], const double wo[3], double T[3], double B[3], double V[3]) {
  frame_of(n, T, B);
  V[0] = wo[0] * T[0] + wo[1] * T[1] + wo[2] * T[2];
  V[1] = wo[0] * B[0] + wo[1] * B[1] + wo[2] * B[2];
  V[2] = wo[0] * n[0] + wo[1] * n[1] + wo[2] * n[2];
  if (V[2] < 1e-4) V[2] = 1e-4;
  normalize3(V);
}
inline double ggx_pdf_local(double alpha, const double V[3], const double L[3]) {
  double H[3] = {V[0] + L[0], V[1] + L[1], V[2] + L[2]};
  normalize3(H);
  if (H[2] <= 0.0) return 0.0;
  const double k = alpha * alpha;
  const double dd = H[2] * H[2] * (k - 1.0) + 1.0;
  const double D = k / (kPi * dd * dd);
  const double G1 = 2.0 * V[2] / (V[2] + std::sqrt(k + (1.0 - k) * V[2] * V[2]));
  return G1 * D / (4.0 * V[2]);                 // D_vis(H) / (4 V.H), D_vis = G1 max(V.H, 0) D / V.z
}
inline void ggx_sample_local(double alpha, const double V[3], double u1, double u2, double L[3]) {
  double Vh[3] = {alpha * V[0], alpha * V[1], V[2]};
  normalize3(Vh);
  double T1[3] = {1.0, 0.0, 0.0};
  const double lensq = Vh[0] * Vh[0] + Vh[1] * Vh[1];
  if (lensq > 1e-14) { const double inv = 1.0 / std::sqrt(lensq); T1[0] = -Vh[1] * inv; T1[1] = Vh[0] * inv; T1[2] = 0.0; }
  const double T2[3] = {Vh[1] * T1[2] - Vh[2] * T1[1], Vh[2] * T1[0] - Vh[0] * T1[2], Vh[0] * T1[1] - Vh[1] * T1[0]};
  const double r = std::sqrt(u1), phi = 2.0 * kPi * u2;
  const double t1 = r * std::cos(phi);
  double t2 = r * std::sin(phi);
  const double s = 0.5 * (1.0 + Vh[2]);
  const double q = 1.0 - t1 * t1;
  t2 = (1.0 - s) * std::sqrt(q > 0.0 ? q : 0.0) + s * t2;
  const double rem = 1.0 - t1 * t1 - t2 * t2;
  const double t3 = std::sqrt(rem > 0.0 ? rem : 0.0);
  double Nh[3] = {t1 * T1[0] + t2 * T2[0] + t3 * Vh[0], t1 * T1[1] + t2 * T2[1] + t3 * Vh[1], t1 * T1[2] + t2 * T2[2] + t3 * Vh[2]};
  double Ne[3] = {alpha * Nh[0], alpha * Nh[1], Nh[2] > 0.0 ? Nh[2] : 0.0};
  normalize3(Ne);
  const double vd = V[0] * Ne[0] + V[1] * Ne[1] + V[2] * Ne[2];
  L[0] = 2.0 * vd * Ne[0] - V[0]; L[1] = 2.0 * vd * Ne[1] - V[1]; L[2] = 2.0 * vd * Ne[2] - V[2];
}

}  // namespace

extern "C" {

uint32_t ors_rng_bits(uint64_t seed, uint64_t row, uint32_t sample, uint32_t dim) { return rng_bits(rng_prefix(seed, row), sample, dim); }
float ors_rng_uniform(uint64_t seed, uint64_t row, uint32_t sample, uint32_t dim) { return rng_uniform(rng_prefix(seed, row), sample, dim); }

void ors_light_tables(const float* env, uint32_t He, uint32_t We, double* pmf, float* cdf) {
  std::vector<double> p; std::vector<float> c;
  build_light_tables(env, He, We, p, c);
  for (size_t k = 0; k < p.size(); ++k) { pmf[k] = p[k]; cdf[k] = c[k]; }
}
void ors_light_pdf(const float* env, uint32_t He, uint32_t We, const double* dirs, uint64_t M, double* out) {
  std::vector<double> p; std::vector<float> c;
  build_light_tables(env, He, We, p, c);
  for (uint64_t m = 0; m < M; ++m) out[m] = light_pdf(p, He, We, dirs + 3 * m);
}
void ors_ggx_pdf(const double* n, const double* rough, const double* wo, const double* wi, uint64_t M, double* out) {
  for (uint64_t m = 0; m < M; ++m) {
    double T[3], B[3], V[3];
    local_view(n + 3 * m, wo + 3 * m, T, B, V);
    const double* w = wi + 3 * m; const double* nn = n + 3 * m;
    const double L[3] = {w[0] * T[0] + w[1] * T[1] + w[2] * T[2], w[0] * B[0] + w[1] * B[1] + w[2] * B[2], w[0] * nn[0] + w[1] * nn[1] + w[2] * nn[2]};
    out[m] = ggx_pdf_local(rough[m] * rough[m], V, L);
  }
}
void ors_ggx_sample(const double* n, const double* rough, const double* wo, const double* u, uint64_t M, double* wi) {
  for (uint64_t m = 0; m < M; ++m) {
    double T[3], B[3], V[3], L[3];
    const double* nn = n + 3 * m;
    local_view(nn, wo + 3 * m, T, B, V);
    ggx_sample_local(rough[m] * rough[m], V, u[2 * m], u[2 * m + 1], L);
    for (int d = 0; d < 3; ++d) wi[3 * m + d] = L[0] * T[d] + L[1] * B[d] + L[2] * nn[d];
  }
}

// MIS direction set of PAPER.md:122: per point, sample s < spp gives a light ray (slot 2s) and a GGX-VNDF ray (slot 2s+1); every
// ray carries the balance-heuristic pdf (p_light + p_ggx) / 2.  brdf [N,7] = n(3) a(3) r(1); texel [N,spp] = chosen env texel.
void ors_sample_mis(const float* env, uint32_t He, uint32_t We, const float* brdf, const float* wo, uint64_t N, uint32_t spp,
                    uint64_t seed, double* dir, double* pdf, uint32_t* texel) {
  std::vector<double> pmf; std::vector<float> cdf;
  build_light_tables(env, He, We, pmf, cdf);
  const uint32_t ntex = He * We;
  const float inv_spp = 1.0f / (float)spp;
  for (uint64_t i = 0; i < N; ++i) {
    const uint32_t pre = rng_prefix(seed, i);
    const double n[3] = {brdf[7 * i], brdf[7 * i + 1], brdf[7 * i + 2]};
    const double w_o[3] = {wo[3 * i], wo[3 * i + 1], wo[3 * i + 2]};
    const double alpha = (double)brdf[7 * i + 6] * (double)brdf[7 * i + 6];
    double T[3], B[3], V[3];
    local_view(n, w_o, T, B, V);
    for (uint32_t s = 0; s < spp; ++s) {
      double* dl = dir + (i * 2 * spp + 2 * s) * 3;
      double* dg = dl + 3;
      {  // light ray: stratified CDF inversion (fp32 decision), jittered inside the texel
        const float u0 = ((float)s + rng_uniform(pre, s, 0)) * inv_spp;
        uint32_t lo = 0, hi = ntex - 1;                        // first k with cdf[k] > u0
        while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (cdf[mid] > u0) hi = mid; else lo = mid + 1; }
        if (texel) texel[i * spp + s] = lo;
        const uint32_t r = lo / We, c = lo % We;
        const double theta = kPi * ((double)r + (double)rng_uniform(pre, s, 1)) / He;
        const double phi = 2.0 * kPi * ((double)c + (double)rng_uniform(pre, s, 2)) / We - kPi;
        dl[0] = std::sin(theta) * std::cos(phi); dl[1] = std::sin(theta) * std::sin(phi); dl[2] = std::cos(theta);
      }
      {  // GGX visible-normal ray
        double L[3];
        ggx_sample_local(alpha, V, (double)rng_uniform(pre, s, 3), (double)rng_uniform(pre, s, 4), L);
        for (int d = 0; d < 3; ++d) dg[d] = L[0] * T[d] + L[1] * B[d] + L[2] * n[d];
      }
      for (int q = 0; q < 2; ++q) {
        const double* w = q ? dg : dl;
        const double Lw[3] = {w[0] * T[0] + w[1] * T[1] + w[2] * T[2], w[0] * B[0] + w[1] * B[1] + w[2] * B[2], w[0] * n[0] + w[1] * n[1] + w[2] * n[2]};
        pdf[i * 2 * spp + 2 * s + q] = 0.5 * (light_pdf(pmf, He, We, w) + ggx_pdf_local(alpha, V, Lw));
      }
    }
  }
}

// Stratified sets: Sa x Sb jittered strata per row.  normal != NULL: cosine-weighted hemisphere about
// normal[row] (pdf cos/pi); normal == NULL: whole sphere (pdf 1/4pi).  Stratum (a, b) -> slot a * Sb + b.
void ors_sample_stratified(const float* normal, uint64_t rows, uint32_t Sa, uint32_t Sb, uint64_t seed, double* dir, double* pdf) {
  for (uint64_t i = 0; i < rows; ++i) {
    const uint32_t pre = rng_prefix(seed, i);
    for (uint32_t a = 0; a < Sa; ++a)
      for (uint32_t b = 0; b < Sb; ++b) {
        const uint32_t s = a * Sb + b;
        const double u = ((double)a + (double)rng_uniform(pre, s, 0)) / Sa;
        const double v = ((double)b + (double)rng_uniform(pre, s, 1)) / Sb;
        double* d = dir + (i * Sa * Sb + s) * 3;
        const double phi = 2.0 * kPi * v;
        if (normal) {
          const double n[3] = {normal[3 * i], normal[3 * i + 1], normal[3 * i + 2]};
          double T[3], B[3];
          frame_of(n, T, B);
          const double r = std::sqrt(u), z = std::sqrt(1.0 - u);
          const double lx = r * std::cos(phi), ly = r * std::sin(phi);
          for (int q = 0; q < 3; ++q) d[q] = lx * T[q] + ly * B[q] + z * n[q];
          pdf[i * Sa * Sb + s] = z / kPi;
        } else {
          const double z = 1.0 - 2.0 * u, r = std::sqrt(1.0 - z * z > 0.0 ? 1.0 - z * z : 0.0);
          d[0] = r * std::cos(phi); d[1] = r * std::sin(phi); d[2] = z;
          pdf[i * Sa * Sb + s] = 1.0 / (4.0 * kPi);
        }
      }
  }
}

}  // extern "C"
