// oracle/hashrender_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU statement of what the recursively executed hash-grid renderer of
// "Baking Relightable NeRF for Real-time Direct/Indirect Illumination Rendering" (arXiv 2409.10327)
// computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may call it.  It shares NO code, header, table or constant with paper_2409_10327_b200/ (the CUDA
// path) and never includes include/hashrender.h.
//
// The method is not a fast route to a separately defined exact result (H, B, I are learned functions,
// Eq. 1 is an MC estimator over a GIVEN direction set), so the oracle is the algorithm itself, step by
// step in the paper's order and notation, in double precision -- except the index path of the encoder,
// which is defined in fp32 so that integer outputs are bit-comparable (reading Q4).
// Every function cites the passage it follows (PAPER.md = /root/reference/PAPER.md) and, where the
// paper is silent, the DESIGN.md reading (Qn) it takes.
//
// Pins (tests/test_oracle_pins.py): hash closed-form known answers, dense-index bijection, corner
// brute force, vertex reproduction, partition of unity, affine reproduction, MLP vs float64 matmul,
// output-map ranges, env texel-centre/constant/wrap, BRDF reciprocity + GGX normalisation + Lambert,
// closed forms a*L, indirect==0 when V==1, a*a'*L, and an independent literal-recursive re-evaluation.
// "Parity with the authors' trained renderer" is PARITY UNPINNED (no weights/datasets exist here).
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

const double kPi = 3.14159265358979323846;

struct OrConfig {            // mirrored field by field in oracle/oracle.py (ctypes)
  uint32_t L, F, log2_T;
  const uint32_t* res;       // [L] integer level resolutions N_l (reading Q2: given, not recomputed)
  uint32_t hidden;           // 64
  float near_t, far_t;       // 0.05, 1.5
  float rough_min;           // 0.09
  float fresnel_f0;          // 0.04
  uint32_t vis_mode;         // 0 soft sigma(z_v), 1 hard [z_v > 0]  (Q14)
  uint32_t brdf_model;       // 0 Lambert, 1 simplified Disney      (Q21)
  float albedo_scale[3];     // PAPER.md:342 (caller-supplied multiplier)
  uint32_t He, We;           // env map size
};

struct OrDirset {            // a direction set (Q19, Q29): dir[.,S,3], pdf[.,S], optional Lin[.,S,3]
  const float* dir; const float* pdf; const float* Lin;
  uint32_t S; uint64_t point_stride;   // elements of `dir` between points; 0 = one shared set
};

inline const float* dir_of(const OrDirset& d, uint64_t i, uint32_t s) { return d.dir + i * d.point_stride + 3ull * s; }
inline float pdf_of(const OrDirset& d, uint64_t i, uint32_t s) { return d.pdf[i * (d.point_stride / 3) + s]; }
inline const float* lin_of(const OrDirset& d, uint64_t i, uint32_t s) { return d.Lin ? d.Lin + i * d.point_stride + 3ull * s : nullptr; }

// ---- step 2: hash-grid encoder H ("multi-level tables as InstantNGP [14]") -------------
// Spatial hash of [14] (reading Q1): XOR of per-axis uint32 products with primes (1, 2654435761,
// 805459861), wrapping multiplies, modulo T = 2^log2_T.
inline uint32_t hash_index(uint32_t cx, uint32_t cy, uint32_t cz, uint32_t log2_T) {
  uint32_t h = (cx * 1u) ^ (cy * 2654435761u) ^ (cz * 805459861u);
  return h & ((1u << log2_T) - 1u);
}
// Level l is dense iff (N_l+1)^3 <= T (64-bit compare), else hashed (reading Q3).
inline bool level_is_dense(uint32_t Nl, uint32_t log2_T) {
  uint64_t v = (uint64_t)Nl + 1; return v * v * v <= (1ull << log2_T);
}
inline uint32_t grid_index(uint32_t cx, uint32_t cy, uint32_t cz, uint32_t Nl, uint32_t log2_T) {
  if (level_is_dense(Nl, log2_T)) return cx + cy * (Nl + 1) + cz * (Nl + 1) * (Nl + 1);
  return hash_index(cx, cy, cz, log2_T);
}

// f = H(x): per level, p = fl32(clamp(x,0,1) * fl32(N_l)) (ONE fp32 multiply; Q4, Q6), c0 = min(floor p,
// N_l-1) (Q7), w = p - c0 (exact in fp32); 8 corners c0 + (b0,b1,b2), corner number b0+2 b1+4 b2;
// trilinear weight prod_d (b_d ? w_d : 1-w_d); f[l*F+j] = sum_c weight_c * tab[l][idx_c][j] (Q9).
void encode_point(const OrConfig& c, const float* tables, const float x[3], double* feat, uint32_t* idx, float* wout) {
  const uint64_t T = 1ull << c.log2_T;
  for (uint32_t l = 0; l < c.L; ++l) {
    const uint32_t Nl = c.res[l];
    uint32_t c0[3]; float w[3];
    for (int d = 0; d < 3; ++d) {
      float xc = x[d]; if (!(xc >= 0.0f)) xc = 0.0f; if (xc > 1.0f) xc = 1.0f;
      volatile float p = xc * (float)Nl;                  // volatile: forbid fusing/extended precision
      int fl = (int)std::floor((float)p);
      if (fl > (int)Nl - 1) fl = (int)Nl - 1;
      c0[d] = (uint32_t)fl;
      w[d] = (float)p - (float)fl;
      if (wout) wout[(l * 3) + d] = w[d];
    }
    for (uint32_t j = 0; j < c.F; ++j) feat[l * c.F + j] = 0.0;
    for (uint32_t corner = 0; corner < 8; ++corner) {
      const uint32_t b0 = corner & 1, b1 = (corner >> 1) & 1, b2 = (corner >> 2) & 1;
      const uint32_t id = grid_index(c0[0] + b0, c0[1] + b1, c0[2] + b2, Nl, c.log2_T);
      if (idx) idx[l * 8 + corner] = id;
      const double wt = (b0 ? (double)w[0] : 1.0 - (double)w[0]) *
                        (b1 ? (double)w[1] : 1.0 - (double)w[1]) *
                        (b2 ? (double)w[2] : 1.0 - (double)w[2]);
      const float* row = tables + ((uint64_t)l * T + id) * c.F;
      for (uint32_t j = 0; j < c.F; ++j) feat[l * c.F + j] += wt * (double)row[j];
    }
  }
}

// ---- steps 3/4: the two 3-layer MLPs ("3 layers in total with hidden dimensions 64") ----
// in -> hidden -> hidden -> out, ReLU on hidden layers (Q10), biases on every layer (Q11).
// Blob: W1[h][in], b1[h], W2[h][h], b2[h], W3[out][h], b3[out].
void mlp3(const float* blob, uint32_t d_in, uint32_t h, uint32_t d_out, const double* in, double* out) {
  const float* W1 = blob; const float* b1 = W1 + (size_t)h * d_in;
  const float* W2 = b1 + h; const float* b2 = W2 + (size_t)h * h;
  const float* W3 = b2 + h; const float* b3 = W3 + (size_t)d_out * h;
  std::vector<double> h1(h), h2(h);
  for (uint32_t j = 0; j < h; ++j) {
    double a = (double)b1[j];
    for (uint32_t k = 0; k < d_in; ++k) a += (double)W1[(size_t)j * d_in + k] * in[k];
    h1[j] = a > 0.0 ? a : 0.0;
  }
  for (uint32_t j = 0; j < h; ++j) {
    double a = (double)b2[j];
    for (uint32_t k = 0; k < h; ++k) a += (double)W2[(size_t)j * h + k] * h1[k];
    h2[j] = a > 0.0 ? a : 0.0;
  }
  for (uint32_t j = 0; j < d_out; ++j) {
    double a = (double)b3[j];
    for (uint32_t k = 0; k < h; ++k) a += (double)W3[(size_t)j * h + k] * h2[k];
    out[j] = a;
  }
}
inline double sigmoid(double z) { return 1.0 / (1.0 + std::exp(-z)); }

// n, a, r = B(f); output maps of PAPER.md:114: n/||n||, sigma(a), 0.09 + sigma(r)*0.91.
// Channel order [n0 n1 n2 a0 a1 a2 r] (Q12); ||n|| guarded by 1e-12; albedo_scale from PAPER.md:342.
void decode_point(const OrConfig& c, const float* brdf_w, const double* feat, double brdf[7]) {
  double o[7];
  mlp3(brdf_w, c.L * c.F, c.hidden, 7, feat, o);
  double nn = std::sqrt(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]); if (nn < 1e-12) nn = 1e-12;
  for (int d = 0; d < 3; ++d) brdf[d] = o[d] / nn;
  for (int d = 0; d < 3; ++d) brdf[3 + d] = sigmoid(o[3 + d]) * (double)c.albedo_scale[d];
  brdf[6] = (double)c.rough_min + sigmoid(o[6]) * (1.0 - (double)c.rough_min);
}

// v, t = I(f, omega): input [f ; omega] (Q13); o = (z_v, z_t);
// v = sigma(z_v) (soft) or [z_v > 0] (hard; Q14, PAPER.md:110 binarises at 0.5);
// d = min(softplus(z_t), 1) ("clamp all outputs to 1 (corresponding to far)"),
// t = near + d (far - near) (min-max normalisation; Q15).
void irt_point(const OrConfig& c, const float* irt_w, const double* feat, const float omega[3],
               double* v, double* zv, double* t) {
  const uint32_t D = c.L * c.F;
  std::vector<double> in(D + 3);
  for (uint32_t k = 0; k < D; ++k) in[k] = feat[k];
  for (int d = 0; d < 3; ++d) in[D + d] = (double)omega[d];
  double o[2];
  mlp3(irt_w, D + 3, c.hidden, 2, in.data(), o);
  *zv = o[0];
  *v = c.vis_mode ? (o[0] > 0.0 ? 1.0 : 0.0) : sigmoid(o[0]);
  double sp = o[1] > 30.0 ? o[1] : std::log1p(std::exp(o[1]));
  double d = sp < 1.0 ? sp : 1.0;
  *t = (double)c.near_t + d * ((double)c.far_t - (double)c.near_t);
}

// ---- step 5: secondary hit x' = x + t*omega, clamped to [0,1]^3 (Q6), no offset (Q20),
// rounded ONCE to fp32 before it is encoded.
void secondary_hit(const float x[3], const float omega[3], double t, float xs[3]) {
  for (int d = 0; d < 3; ++d) {
    double v = (double)x[d] + t * (double)omega[d];
    if (v < 0.0) v = 0.0; if (v > 1.0) v = 1.0;
    xs[d] = (float)v;
  }
}

// ---- step 6: image-based lighting lookup ("pixels of the environment map are interpolated")
// Equirect (Q25): z-up, theta = acos(omega_z) from +z, phi = atan2(omega_y, omega_x), texel centres at
// half-integers: u = (phi/2pi + 1/2) We - 1/2, s = (theta/pi) He - 1/2; bilinear; wrap in u, clamp in s.
void env_lookup(const OrConfig& c, const float* env, const double w[3], double rgb[3]) {
  double wz = w[2] < -1.0 ? -1.0 : (w[2] > 1.0 ? 1.0 : w[2]);
  const double theta = std::acos(wz), phi = std::atan2(w[1], w[0]);
  const double u = (phi / (2.0 * kPi) + 0.5) * c.We - 0.5;
  const double s = (theta / kPi) * c.He - 0.5;
  const double u0 = std::floor(u), s0 = std::floor(s);
  const double fu = u - u0, fs = s - s0;
  const long We = c.We, He = c.He;
  long x0 = ((long)u0 % We + We) % We, x1 = (x0 + 1) % We;
  long y0 = (long)s0, y1 = y0 + 1;
  if (y0 < 0) y0 = 0; if (y0 > He - 1) y0 = He - 1;
  if (y1 < 0) y1 = 0; if (y1 > He - 1) y1 = He - 1;
  for (int ch = 0; ch < 3; ++ch) {
    const double e00 = env[(y0 * We + x0) * 3 + ch], e01 = env[(y0 * We + x1) * 3 + ch];
    const double e10 = env[(y1 * We + x0) * 3 + ch], e11 = env[(y1 * We + x1) * 3 + ch];
    rgb[ch] = (1.0 - fs) * ((1.0 - fu) * e00 + fu * e01) + fs * ((1.0 - fu) * e10 + fu * e11);
  }
}

// ---- step 7: BRDF (PAPER.md:62 simplified Disney; PAPER.md:122 alpha = r^2, k = alpha^2;
// PAPER.md:128 Schlick Fresnel + correlated Smith; PAPER.md:252 F0 = 0.04; reading Q21).
// Returns f_r * NoL / pdf per channel WITHOUT the radiance factor; 0 if NoL <= 0 or pdf <= 0 (Q22, Q23).
void brdf_cos_over_pdf(const OrConfig& c, const double brdf[7], const double wi[3], const double wo[3],
                       double pdf, double out[3]) {
  out[0] = out[1] = out[2] = 0.0;
  const double* n = brdf; const double* a = brdf + 3; const double r = brdf[6];
  const double NoL = n[0] * wi[0] + n[1] * wi[1] + n[2] * wi[2];
  if (!(NoL > 0.0) || !(pdf > 0.0)) return;
  double spec = 0.0;
  if (c.brdf_model == 1) {
    double NoV = n[0] * wo[0] + n[1] * wo[1] + n[2] * wo[2]; if (NoV < 1e-4) NoV = 1e-4;
    double h[3] = {wi[0] + wo[0], wi[1] + wo[1], wi[2] + wo[2]};
    double hn = std::sqrt(h[0] * h[0] + h[1] * h[1] + h[2] * h[2]); if (hn < 1e-12) hn = 1e-12;
    for (int d = 0; d < 3; ++d) h[d] /= hn;
    double NoH = n[0] * h[0] + n[1] * h[1] + n[2] * h[2]; if (NoH < 0.0) NoH = 0.0;
    double VoH = wo[0] * h[0] + wo[1] * h[1] + wo[2] * h[2]; if (VoH < 0.0) VoH = 0.0;
    const double alpha = r * r, k = alpha * alpha;
    const double dd = NoH * NoH * (k - 1.0) + 1.0;
    const double D = k / (kPi * dd * dd);
    const double F = (double)c.fresnel_f0 + (1.0 - (double)c.fresnel_f0) * std::pow(1.0 - VoH, 5.0);
    const double Gv = 0.5 / (NoL * std::sqrt(NoV * NoV * (1.0 - k) + k) + NoV * std::sqrt(NoL * NoL * (1.0 - k) + k));
    spec = D * F * Gv;
  }
  for (int ch = 0; ch < 3; ++ch) out[ch] = (a[ch] / kPi + spec) * NoL / pdf;
}

void incoming(const OrConfig& c, const float* env, const OrDirset& ds, uint64_t i, uint32_t s, double L[3]) {
  const float* lin = lin_of(ds, i, s);
  if (lin) { L[0] = lin[0]; L[1] = lin[1]; L[2] = lin[2]; return; }
  const float* w = dir_of(ds, i, s);
  const double wd[3] = {(double)w[0], (double)w[1], (double)w[2]};
  env_lookup(c, env, wd, L);
}

// ---- step 8: outgoing radiance L'_o at a secondary point x': f' = H(x'),
// a', r', n' = B(f'), omega_o' = -omega_j (Q17), v' = I(f', omega'_k) (Q18), Eq. 1 over the tertiary set,
// no further recursion ("limited to 2-bounce").  `tert_point` = row of the tertiary set.
void secondary_radiance(const OrConfig& c, const float* tables, const float* brdf_w, const float* irt_w,
                        const float* env, const float xs[3], const float omega_j[3], const OrDirset& tert,
                        uint64_t tert_point, double delta, double Lo[3], double flip[3]) {
  const uint32_t D = c.L * c.F;
  std::vector<double> f(D);
  encode_point(c, tables, xs, f.data(), nullptr, nullptr);
  double brdf[7];
  decode_point(c, brdf_w, f.data(), brdf);
  const double wo[3] = {-(double)omega_j[0], -(double)omega_j[1], -(double)omega_j[2]};
  Lo[0] = Lo[1] = Lo[2] = 0.0; flip[0] = flip[1] = flip[2] = 0.0;
  for (uint32_t k = 0; k < tert.S; ++k) {
    const float* w = dir_of(tert, tert_point, k);
    double v, zv, t;
    irt_point(c, irt_w, f.data(), w, &v, &zv, &t);
    double L[3], g[3];
    incoming(c, env, tert, tert_point, k, L);
    const double wd[3] = {(double)w[0], (double)w[1], (double)w[2]};
    brdf_cos_over_pdf(c, brdf, wd, wo, (double)pdf_of(tert, tert_point, k), g);
    for (int ch = 0; ch < 3; ++ch) {
      Lo[ch] += v * L[ch] * g[ch];
      if (c.vis_mode && std::fabs(zv) < delta) flip[ch] += std::fabs(L[ch] * g[ch]);
    }
  }
  for (int ch = 0; ch < 3; ++ch) { Lo[ch] /= (double)tert.S; flip[ch] /= (double)tert.S; }   // Q24
}

}  // namespace

extern "C" {

uint32_t or_hash_index(uint32_t cx, uint32_t cy, uint32_t cz, uint32_t log2_T) { return hash_index(cx, cy, cz, log2_T); }
uint32_t or_grid_index(uint32_t cx, uint32_t cy, uint32_t cz, uint32_t Nl, uint32_t log2_T) { return grid_index(cx, cy, cz, Nl, log2_T); }
int or_level_is_dense(uint32_t Nl, uint32_t log2_T) { return level_is_dense(Nl, log2_T) ? 1 : 0; }

// feat[N, L*F] double; idx (nullable) [N, L, 8] uint32; w (nullable) [N, L, 3] float.
void or_encode(const OrConfig* c, const float* tables, const float* x, uint64_t N, double* feat, uint32_t* idx, float* w) {
  const uint32_t D = c->L * c->F;
  for (uint64_t i = 0; i < N; ++i)
    encode_point(*c, tables, x + 3 * i, feat + i * D, idx ? idx + i * c->L * 8 : nullptr, w ? w + i * c->L * 3 : nullptr);
}

void or_mlp3(const float* blob, uint32_t d_in, uint32_t h, uint32_t d_out, const double* in, uint64_t N, double* out) {
  for (uint64_t i = 0; i < N; ++i) mlp3(blob, d_in, h, d_out, in + i * d_in, out + i * d_out);
}

void or_decode(const OrConfig* c, const float* brdf_w, const double* feat, uint64_t N, double* brdf) {
  const uint32_t D = c->L * c->F;
  for (uint64_t i = 0; i < N; ++i) decode_point(*c, brdf_w, feat + i * D, brdf + i * 7);
}

// vis, zv, t: [N,S] double; xsec (nullable): [N,S,3] float (step 5).
void or_trace(const OrConfig* c, const float* irt_w, const float* x, const double* feat, uint64_t N,
              const OrDirset* ds, double* vis, double* zv, double* t, float* xsec) {
  const uint32_t D = c->L * c->F;
  for (uint64_t i = 0; i < N; ++i)
    for (uint32_t s = 0; s < ds->S; ++s) {
      const float* w = dir_of(*ds, i, s);
      double v, z, tt;
      irt_point(*c, irt_w, feat + i * D, w, &v, &z, &tt);
      vis[i * ds->S + s] = v; zv[i * ds->S + s] = z; t[i * ds->S + s] = tt;
      if (xsec) secondary_hit(x + 3 * i, w, tt, xsec + (i * ds->S + s) * 3);
    }
}

void or_env_lookup(const OrConfig* c, const float* env, const double* dirs, uint64_t M, double* rgb) {
  for (uint64_t i = 0; i < M; ++i) env_lookup(*c, env, dirs + 3 * i, rgb + 3 * i);
}

// f_r (without cos / pdf): evaluates brdf_cos_over_pdf and undoes the NoL/pdf factor for NoL > 0.
void or_brdf_eval(const OrConfig* c, const double* brdf, const double* wi, const double* wo, double* fr) {
  double g[3];
  brdf_cos_over_pdf(*c, brdf, wi, wo, 1.0, g);
  const double NoL = brdf[0] * wi[0] + brdf[1] * wi[1] + brdf[2] * wi[2];
  for (int ch = 0; ch < 3; ++ch) fr[ch] = NoL > 0.0 ? g[ch] / NoL : 0.0;
}

// step 9 on ONE direction set (Eq. 1 with Eq. 2 per direction):
// rgb = 1/S sum_s [ (terms&1) v L_i + (terms&2) (1-v) Lind ] f_r NoL / p.   vis [N,S]; Lind nullable [N,S,3].
void or_shade(const OrConfig* c, const float* env, const double* brdf, const float* wo, uint64_t N,
              const OrDirset* ds, const double* vis, const double* Lind, uint32_t terms, double* rgb) {
  for (uint64_t i = 0; i < N; ++i) {
    const double wod[3] = {(double)wo[3 * i], (double)wo[3 * i + 1], (double)wo[3 * i + 2]};
    double acc[3] = {0, 0, 0};
    for (uint32_t s = 0; s < ds->S; ++s) {
      const float* w = dir_of(*ds, i, s);
      const double wd[3] = {(double)w[0], (double)w[1], (double)w[2]};
      double g[3], L[3] = {0, 0, 0};
      brdf_cos_over_pdf(*c, brdf + 7 * i, wd, wod, (double)pdf_of(*ds, i, s), g);
      if (terms & 1) incoming(*c, env, *ds, i, s, L);
      const double v = vis[i * ds->S + s];
      for (int ch = 0; ch < 3; ++ch) {
        double Lt = (terms & 1) ? v * L[ch] : 0.0;
        if ((terms & 2) && Lind) Lt += (1.0 - v) * Lind[(i * ds->S + s) * 3 + ch];
        acc[ch] += Lt * g[ch];
      }
    }
    for (int ch = 0; ch < 3; ++ch) rgb[3 * i + ch] = acc[ch] / (double)ds->S;
  }
}

// Whole frame (steps 1-9).  brdf_ext nullable [N,7] double-widened by caller as float (Q30: NULL => B(H(x))).
// flags: 1 DIRECT, 2 SHADOW, 4 INDIRECT.  mask nullable (Q27).  flipbound (nullable) [N,3]: Q33 bound with
// threshold `delta` on |z_v| (hard mode only).  stats (nullable) [2]: {#secondary points, #of them with a clamped coordinate}.
void or_render_frame(const OrConfig* c, const float* tables, const float* brdf_w, const float* irt_w, const float* env,
                     uint64_t N, const float* x, const float* brdf_ext, const float* wo, const uint8_t* mask,
                     const OrDirset* direct, const OrDirset* secondary, const OrDirset* tertiary, uint32_t flags,
                     double delta, double* rgb, double* flipbound, uint64_t* stats) {
  const uint32_t D = c->L * c->F;
  std::vector<double> f(D);
  if (stats) stats[0] = stats[1] = 0;
  for (uint64_t i = 0; i < N; ++i) {
    double* out = rgb + 3 * i;
    out[0] = out[1] = out[2] = 0.0;
    double fb[3] = {0, 0, 0};
    if (mask && !mask[i]) { if (flipbound) { flipbound[3 * i] = flipbound[3 * i + 1] = flipbound[3 * i + 2] = 0.0; } continue; }
    encode_point(*c, tables, x + 3 * i, f.data(), nullptr, nullptr);
    double brdf[7];
    if (brdf_ext) for (int k = 0; k < 7; ++k) brdf[k] = (double)brdf_ext[7 * i + k];
    else decode_point(*c, brdf_w, f.data(), brdf);
    const double wod[3] = {(double)wo[3 * i], (double)wo[3 * i + 1], (double)wo[3 * i + 2]};
    if ((flags & 1) && direct && direct->S) {                 // direct term of Eq. 1
      double acc[3] = {0, 0, 0};
      for (uint32_t s = 0; s < direct->S; ++s) {
        const float* w = dir_of(*direct, i, s);
        double v = 1.0, zv = 1e30, t;
        if (flags & 2) irt_point(*c, irt_w, f.data(), w, &v, &zv, &t);     // shadow visibility
        double L[3], g[3];
        incoming(*c, env, *direct, i, s, L);
        const double wd[3] = {(double)w[0], (double)w[1], (double)w[2]};
        brdf_cos_over_pdf(*c, brdf, wd, wod, (double)pdf_of(*direct, i, s), g);
        for (int ch = 0; ch < 3; ++ch) {
          acc[ch] += v * L[ch] * g[ch];
          if (c->vis_mode && std::fabs(zv) < delta) fb[ch] += std::fabs(L[ch] * g[ch]) / (double)direct->S;
        }
      }
      for (int ch = 0; ch < 3; ++ch) out[ch] += acc[ch] / (double)direct->S;
    }
    if ((flags & 4) && secondary && secondary->S) {           // (1 - V) L'_o term of Eq. 2
      double acc[3] = {0, 0, 0};
      for (uint32_t j = 0; j < secondary->S; ++j) {
        const float* w = dir_of(*secondary, i, j);
        double v, zv, t;
        irt_point(*c, irt_w, f.data(), w, &v, &zv, &t);
        float xs[3];
        secondary_hit(x + 3 * i, w, t, xs);
        if (stats) {
          stats[0]++;
          if (xs[0] <= 0.f || xs[0] >= 1.f || xs[1] <= 0.f || xs[1] >= 1.f || xs[2] <= 0.f || xs[2] >= 1.f) stats[1]++;
        }
        double Lo[3], fl[3], g[3];
        secondary_radiance(*c, tables, brdf_w, irt_w, env, xs, w, *tertiary,
                           tertiary->point_stride ? i * secondary->S + j : 0, delta, Lo, fl);
        const double wd[3] = {(double)w[0], (double)w[1], (double)w[2]};
        brdf_cos_over_pdf(*c, brdf, wd, wod, (double)pdf_of(*secondary, i, j), g);
        for (int ch = 0; ch < 3; ++ch) {
          acc[ch] += (1.0 - v) * Lo[ch] * g[ch];
          fb[ch] += (1.0 - v) * fl[ch] * std::fabs(g[ch]) / (double)secondary->S;
          if (c->vis_mode && std::fabs(zv) < delta) fb[ch] += std::fabs(Lo[ch] * g[ch]) / (double)secondary->S;
        }
      }
      for (int ch = 0; ch < 3; ++ch) out[ch] += acc[ch] / (double)secondary->S;
    }
    if (flipbound) for (int ch = 0; ch < 3; ++ch) flipbound[3 * i + ch] = fb[ch];
  }
}

}  // extern "C"
