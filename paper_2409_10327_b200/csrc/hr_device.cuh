// hr_device.cuh -- parameter blocks and per-thread device math shared by the hashrender kernels:
// hash-grid encode, output maps, env lookup, BRDF
// (PAPER.md:62, 122, 128, 252), secondary hit.  fp32 throughout; the index path is kept to
// single IEEE operations (__fmul_rn / __fsub_rn) so integer outputs are bit-exact (Q4).
#pragma once
#include <cuda_fp16.h>
#include <stdint.h>

namespace hr {

constexpr int kMaxL = 16;   // levels
constexpr int kD = 32;      // padded feature width (L*F <= 32, F == 2)
constexpr int kH = 64;      // hidden width

// Device layout of the tables (hashrender_create re-lays them out once): level l starts `off[l]` bytes into `tables` and the row of
// grid vertex (cx, cy, cz) is  (cx ^ cy * pa[l] ^ cz * pb[l]) & pmask[l]  for EVERY level.  Hashed levels: pa, pb = the primes of
// [14], pmask = T - 1, T rows (Q1).  Dense levels: the vertex index is stored with power-of-two strides, pa = 2^b, pb = 2^2b,
// b = ceil(log2(N + 1)), pmask = ~0: the three terms occupy disjoint bits, so the XOR is the sum cx + cy 2^b + cz 2^2b.  One branch-free
// index path serves both kinds, and the two x-neighbours of a cell are ADJACENT rows whenever cx is even (bit 0 of the row is
// bit 0 of cx), so one aligned two-row load brings both (gather8).  The index the ABI exports (hashrender_encode) is still the
// specified one, x + y (N+1) + z (N+1)^2 or the hash (corner_indices).  Levels l >= L are null: res 1, pa = pb = pmask = 0, off = a
// block of zero rows.
// Cell-major levels (l < nblock, the coarsest ones; hashrender_create picks them by a byte budget): the level is stored as N^3 ENTRIES,
// one per grid cell (cx, cy, cz), entry index cx + N (cy + N cz), each the cell's 8 corner rows in corner order b0 + 2 b1 + 4 b2 -- the
// rows the specified index (dense or hashed) names, copied, so values and arithmetic are unchanged.  An entry of fp16 rows is one
// aligned 32-byte sector (ONE 256-bit load), of fp32 rows two sectors (two loads), against 8 one-row loads that touch ~4.5 sectors:
// an SM's L1 passes ONE missing sector per cycle to the L2 (measured with fully divergent loads of any width, 289 G loads/s for the
// chip) and that rate, not arithmetic, bounds the encode, so a level costs one or two sector requests instead of 4.5.
struct GridP {
  uint32_t L, log2_T, dense_mask, f16, nblock;
  uint32_t res[kMaxL];
  uint32_t pa[kMaxL], pb[kMaxL], pmask[kMaxL];
  unsigned long long off[kMaxL];
  const void* tables;       // rows of float2 (f16 == 0) or __half2 (f16 == 1)
  uint32_t l2_hint;         // hashed levels > 2 x L2: their gathers carry an evict-first policy, dense levels evict-last (k_trace_wg)
  uint32_t pair_loads;      // fp16 rows, device copy of the tables L2-resident: x-neighbour pairs come with one two-row load (gather8_h2)
};
// L2 eviction policies for tables far larger than the L2 (BASELINE configs[4], T = 2^24): the hashed levels are a random stream over
// hundreds of MB that no cache can hold, the dense levels are ~70 MB that every point reads.  Hashed rows are fetched evict-first
// and dense rows evict-last, so the stream does not push the dense levels out.  Measured with k_trace_wg at 2^24 points: T = 2^24
// (448 MB of hashed levels) 13.5 -> 12.6 ms; evict-first alone 12.7, evict-last alone 13.4 (no effect); at T = 2^22 (128 MB of
// hashed levels, about the size of the L2) the hint LOSES, 11.45 -> 12.15 ms, so it is applied only when the hashed levels exceed
// twice the L2 (hashrender_create).
struct L2Pol { unsigned long long first, last; };
__device__ __forceinline__ L2Pol make_l2pol() {
  L2Pol p;
  asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p.first));
  asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p.last));
  return p;
}
struct EnvP { const float* env; const float4* env4; uint32_t He, We; };     // env4: the same texels padded to RGBA (one 16-byte load each)
struct ShadeP {
  float near_t, far_t, rough_min, f0;
  uint32_t vis_mode, brdf_model;
  float as0, as1, as2;
};
struct DirsetP {
  const float* dir; const float* pdf; const float* Lin;
  uint32_t S; unsigned long long stride;
};
struct FrameP {
  unsigned long long N;
  const float* x; const float* brdf; const float* wo; const uint8_t* mask;
  DirsetP d, s, t;
  uint32_t flags;
};

__device__ __forceinline__ const float* dir_of(const DirsetP& d, unsigned long long i, uint32_t s) {
  return d.dir + i * d.stride + 3ull * s;
}
__device__ __forceinline__ float pdf_of(const DirsetP& d, unsigned long long i, uint32_t s) {
  return __ldg(d.pdf + i * (d.stride / 3ull) + s);
}

// ---- a1/a2: level scale, corner select, spatial hash / dense index ---------------------------------
struct Cell { uint32_t c0[3]; float w[3]; };

__device__ __forceinline__ Cell cell_of(uint32_t N, float x, float y, float z) {
  Cell c;
  const float fn = (float)N;
  const float p[3] = {__fmul_rn(fminf(fmaxf(x, 0.f), 1.f), fn), __fmul_rn(fminf(fmaxf(y, 0.f), 1.f), fn),
                      __fmul_rn(fminf(fmaxf(z, 0.f), 1.f), fn)};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    int fl = min(__float2int_rd(p[d]), (int)N - 1);          // Q7: x == 1 -> c0 = N-1, w = 1
    c.c0[d] = (uint32_t)fl;
    c.w[d] = __fsub_rn(p[d], (float)fl);
  }
  return c;
}

// same for a position already clamped to [0,1]^3 (x' = sec_hit(...) is)
__device__ __forceinline__ Cell cell_of_clamped(uint32_t N, float x, float y, float z) {
  Cell c;
  const float fn = (float)N;
  const float p[3] = {__fmul_rn(x, fn), __fmul_rn(y, fn), __fmul_rn(z, fn)};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    int fl = min(__float2int_rd(p[d]), (int)N - 1);
    c.c0[d] = (uint32_t)fl;
    c.w[d] = __fsub_rn(p[d], (float)fl);
  }
  return c;
}

__device__ __forceinline__ void corner_indices(const Cell& c, uint32_t N, bool dense, uint32_t log2_T, uint32_t (&idx)[8]) {
  if (dense) {                                                // (N+1)^3 <= T (Q3)
    const uint32_t s = N + 1, s2 = s * s;
    const uint32_t base = c.c0[0] + c.c0[1] * s + c.c0[2] * s2;
#pragma unroll
    for (int k = 0; k < 8; ++k) idx[k] = base + (k & 1) + ((k >> 1) & 1) * s + ((k >> 2) & 1) * s2;
  } else {                                                    // hash of [14], primes (1, 2654435761, 805459861) (Q1)
    const uint32_t mask = (1u << log2_T) - 1u;
    const uint32_t hx[2] = {c.c0[0], c.c0[0] + 1u};
    const uint32_t hy0 = c.c0[1] * 2654435761u, hy1 = hy0 + 2654435761u;
    const uint32_t hz0 = c.c0[2] * 805459861u, hz1 = hz0 + 805459861u;
    const uint32_t hyz[4] = {hy0 ^ hz0, hy1 ^ hz0, hy0 ^ hz1, hy1 ^ hz1};
#pragma unroll
    for (int k = 0; k < 8; ++k) idx[k] = (hx[k & 1] ^ hyz[k >> 1]) & mask;
  }
}

// a3: the 8 corner rows of one level, corner number b0 + 2 b1 + 4 b2 (Q9): one index path for dense and hashed levels (address =
// level base + row * row bytes in one mad.wide.u32, read-only path).  fp32 rows: eight independent one-row loads.  fp16 rows: the
// x-neighbour pair comes with one aligned two-row load when cx is even (gather8_h2).
__device__ __forceinline__ void corner_rows(const GridP& g, int l, const uint32_t (&c0)[3], uint32_t (&i0)[4], uint32_t (&i1)[4]) {
  const uint32_t pa = g.pa[l], pb = g.pb[l], pm = g.pmask[l];
  const uint32_t hy0 = c0[1] * pa, hy1 = hy0 + pa, hz0 = c0[2] * pb, hz1 = hz0 + pb;
  const uint32_t h[4] = {hy0 ^ hz0, hy1 ^ hz0, hy0 ^ hz1, hy1 ^ hz1};
#pragma unroll
  for (int j = 0; j < 4; ++j) { i0[j] = (c0[0] ^ h[j]) & pm; i1[j] = ((c0[0] + 1u) ^ h[j]) & pm; }
}
// entry of cell c0 of a cell-major level
__device__ __forceinline__ const uint4* block_entry(const GridP& g, int l, const uint32_t (&c0)[3], uint32_t entry_bytes) {
  const uint32_t N = g.res[l];
  const uint32_t e = c0[0] + N * (c0[1] + N * c0[2]);
  return reinterpret_cast<const uint4*>(reinterpret_cast<const char*>(g.tables) + g.off[l] + (unsigned long long)e * entry_bytes);
}
// one aligned 32-byte sector in ONE load (sm_100 has 256-bit global loads)
__device__ __forceinline__ void ldg_nc32(const uint4* p, uint32_t (&r)[8]) {
  asm("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "l"(p));
}
template <int PAIR = -1>                      // -1: g.pair_loads decides at run time; 0 / 1: the caller's kernel was chosen by it
__device__ __forceinline__ void gather8_h2(const GridP& g, int l, const uint32_t (&c0)[3], uint32_t (&v)[8]) {
  if (l < (int)g.nblock) {                                    // warp-uniform: l is a loop counter
    ldg_nc32(block_entry(g, l, c0, 32u), v);
    return;
  }
  uint32_t i0[4], i1[4];
  corner_rows(g, l, c0, i0, i1);
  const char* lb = reinterpret_cast<const char*>(g.tables) + g.off[l];
  // The aligned 8-byte word of row i0 always holds row i0 ^ 1, and that IS the x-neighbour when cx is even (bit 0 of a row is bit 0
  // of cx on every level): one 8-byte load serves the pair, a predicated one-row load fetches the neighbour for odd cx.  6 loads per
  // level instead of 8 on average; each costs the L1 0.35 cycles (hashrender_probe_gather).  Same box: C3 dense 15.00 -> 14.50 ms,
  // compacted 7.16 -> 7.04, C4 at T = 2^19 4.71 -> 4.64.  (Before the cell-major levels the same idea LOST -- C3 16.7 -> 17.6 -- and
  // for 8-byte fp32 rows it still does, C2 23.05 -> 24.35: the 16-byte pair words cost the split-precision kernel registers it
  // does not have.  gather8_f2 keeps one load per row.)
  // Only while the tables are L2-resident (g.pair_loads, set by hashrender_create): with tables that spill to HBM the same loads
  // LOSE (k_trace_wg at T = 2^22, 2^24 points: 8.56 -> 9.23 ms on one box), and one load per row stays.
  if (PAIR == 0 || (PAIR < 0 && !g.pair_loads)) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      asm("{\n\t.reg .u64 p;\n\tmad.wide.u32 p, %1, 4, %2;\n\tld.global.nc.b32 %0, [p];\n\t}" : "=r"(v[2 * j]) : "r"(i0[j]), "l"(lb));
      asm("{\n\t.reg .u64 p;\n\tmad.wide.u32 p, %1, 4, %2;\n\tld.global.nc.b32 %0, [p];\n\t}" : "=r"(v[2 * j + 1]) : "r"(i1[j]), "l"(lb));
    }
    return;
  }
  const bool odd = c0[0] & 1u;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    uint32_t lo, hi, nb = 0u;
    asm("{\n\t.reg .u64 p;\n\tmad.wide.u32 p, %2, 4, %3;\n\tld.global.nc.v2.b32 {%0, %1}, [p];\n\t}" : "=r"(lo), "=r"(hi) : "r"(i0[j] & ~1u), "l"(lb));
    if (odd) asm("{\n\t.reg .u64 p;\n\tmad.wide.u32 p, %1, 4, %2;\n\tld.global.nc.b32 %0, [p];\n\t}" : "=r"(nb) : "r"(i1[j]), "l"(lb));
    const bool up = i0[j] & 1u;
    v[2 * j] = up ? hi : lo;
    v[2 * j + 1] = odd ? nb : (up ? lo : hi);
  }
}
// the same with an L2 eviction policy per level (hashed: evict-first, dense: evict-last)
__device__ __forceinline__ void gather8_h2_hint(const GridP& g, int l, const uint32_t (&c0)[3], uint32_t (&v)[8], const L2Pol& pol) {
  if (l < (int)g.nblock) { gather8_h2<0>(g, l, c0, v); return; }
  uint32_t i0[4], i1[4];
  corner_rows(g, l, c0, i0, i1);
  const char* lb = reinterpret_cast<const char*>(g.tables) + g.off[l];
  const unsigned long long cp = g.pmask[l] == 0xFFFFFFFFu ? pol.last : pol.first;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    asm("{\n\t.reg .u64 p;\n\tmad.wide.u32 p, %1, 4, %2;\n\tld.global.nc.L2::cache_hint.b32 %0, [p], %3;\n\t}" : "=r"(v[2 * j]) : "r"(i0[j]), "l"(lb), "l"(cp));
    asm("{\n\t.reg .u64 p;\n\tmad.wide.u32 p, %1, 4, %2;\n\tld.global.nc.L2::cache_hint.b32 %0, [p], %3;\n\t}" : "=r"(v[2 * j + 1]) : "r"(i1[j]), "l"(lb), "l"(cp));
  }
}
__device__ __forceinline__ void gather8_f2(const GridP& g, int l, const uint32_t (&c0)[3], float2 (&v)[8]) {
  if (l < (int)g.nblock) {
    const uint4* p = block_entry(g, l, c0, 64u);
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      uint32_t r[8];
      ldg_nc32(p + 2 * j, r);
#pragma unroll
      for (int k = 0; k < 4; ++k) v[4 * j + k] = make_float2(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
    }
    return;
  }
  uint32_t i0[4], i1[4];
  corner_rows(g, l, c0, i0, i1);
  const char* lb = reinterpret_cast<const char*>(g.tables) + g.off[l];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    asm("{\n\t.reg .u64 p;\n\tmad.wide.u32 p, %2, 8, %3;\n\tld.global.nc.v2.f32 {%0, %1}, [p];\n\t}" : "=f"(v[2 * j].x), "=f"(v[2 * j].y) : "r"(i0[j]), "l"(lb));
    asm("{\n\t.reg .u64 p;\n\tmad.wide.u32 p, %2, 8, %3;\n\tld.global.nc.v2.f32 {%0, %1}, [p];\n\t}" : "=f"(v[2 * j + 1].x), "=f"(v[2 * j + 1].y) : "r"(i1[j]), "l"(lb));
  }
}
template <bool F16, int PAIR = -1>
__device__ __forceinline__ void gather8(const GridP& g, int l, const uint32_t (&c0)[3], float2 (&v)[8]) {
  if constexpr (F16) {
    uint32_t r[8];
    gather8_h2<PAIR>(g, l, c0, r);
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = __half22float2(*reinterpret_cast<const __half2*>(&r[k]));
  } else {
    gather8_f2(g, l, c0, v);
  }
}

// a3/a4: gather 8 corners of one level and interpolate.  Corner number b0 + 2 b1 + 4 b2 (Q9).
template <bool F16, int PAIR = -1>
__device__ __forceinline__ float2 encode_level(const GridP& g, int l, float x, float y, float z,
                                               uint32_t* idx_out, float* w_out, const L2Pol* pol = nullptr) {
  const uint32_t N = g.res[l];
  const Cell c = cell_of(N, x, y, z);
  float2 v[8];
  if (F16 && pol) {
    uint32_t r[8];
    gather8_h2_hint(g, l, c.c0, r, *pol);
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = __half22float2(*reinterpret_cast<const __half2*>(&r[k]));
  } else {
    gather8<F16, PAIR>(g, l, c.c0, v);
  }
  if (idx_out) {                                              // the SPECIFIED index (Q1, Q3), not the device row
    uint32_t idx[8];
    corner_indices(c, N, (g.dense_mask >> l) & 1u, g.log2_T, idx);
#pragma unroll
    for (int k = 0; k < 8; ++k) idx_out[k] = idx[k];
  }
  if (w_out) { w_out[0] = c.w[0]; w_out[1] = c.w[1]; w_out[2] = c.w[2]; }
  const float wx[2] = {1.f - c.w[0], c.w[0]}, wy[2] = {1.f - c.w[1], c.w[1]}, wz[2] = {1.f - c.w[2], c.w[2]};
  float2 f = make_float2(0.f, 0.f);
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const float wt = wx[k & 1] * wy[(k >> 1) & 1] * wz[(k >> 2) & 1];
    f.x = fmaf(wt, v[k].x, f.x);
    f.y = fmaf(wt, v[k].y, f.y);
  }
  return f;
}

// f = H(x), zero-padded to kD entries.
template <bool F16>
__device__ __forceinline__ void encode_point(const GridP& g, float x, float y, float z, float (&f)[kD]) {
#pragma unroll
  for (int l = 0; l < kMaxL; ++l) {
    if (l < (int)g.L) {
      const float2 v = encode_level<F16>(g, l, x, y, z, nullptr, nullptr);
      f[2 * l] = v.x; f[2 * l + 1] = v.y;
    } else {
      f[2 * l] = 0.f; f[2 * l + 1] = 0.f;
    }
  }
}

// ---- output maps ------------------------------------------------------------------------------------
__device__ __forceinline__ float sigmoidf_(float z) { return 1.f / (1.f + expf(-z)); }

// o[0..6] raw B outputs -> n/||n||, sigma(a)*scale, rough_min + sigma(r)(1 - rough_min)  (Q12)
__device__ __forceinline__ void brdf_maps(const ShadeP& sp, const float (&o)[8], float (&b)[7]) {
  const float nn = fmaxf(sqrtf(o[0] * o[0] + o[1] * o[1] + o[2] * o[2]), 1e-12f);
  const float inv = 1.f / nn;
  b[0] = o[0] * inv; b[1] = o[1] * inv; b[2] = o[2] * inv;
  b[3] = sigmoidf_(o[3]) * sp.as0; b[4] = sigmoidf_(o[4]) * sp.as1; b[5] = sigmoidf_(o[5]) * sp.as2;
  b[6] = sp.rough_min + sigmoidf_(o[6]) * (1.f - sp.rough_min);
}

// (z_v, z_t) -> v, t  (Q14, Q15).  softplus(z) >= 1 iff z >= ln(e-1), so the clamp
// removes the large-z branch.
__device__ __forceinline__ void irt_maps(const ShadeP& sp, float zv, float zt, float& v, float& t) {
  v = sp.vis_mode ? (zv > 0.f ? 1.f : 0.f) : sigmoidf_(zv);
  const float d = zt > 0.6f ? 1.f : fminf(log1pf(expf(zt)), 1.f);
  t = sp.near_t + d * (sp.far_t - sp.near_t);
}

// a7: x' = clamp(x + t w, 0, 1)  (Q6, Q20)
__device__ __forceinline__ float sec_hit(float x, float t, float w) { return fminf(fmaxf(fmaf(t, w, x), 0.f), 1.f); }

// ---- a9: equirect bilinear env lookup (Q25) ------------------------------------------------
__device__ __forceinline__ float3 env_lookup(const EnvP& e, float wx, float wy, float wz) {
  const float theta = acosf(fminf(fmaxf(wz, -1.f), 1.f));
  const float phi = atan2f(wy, wx);
  const float u = (phi * 0.15915494309189535f + 0.5f) * (float)e.We - 0.5f;
  const float s = (theta * 0.3183098861837907f) * (float)e.He - 0.5f;
  const float u0 = floorf(u), s0 = floorf(s);
  const float fu = u - u0, fs = s - s0;
  const int We = (int)e.We, He = (int)e.He;
  int x0 = (int)u0 % We; if (x0 < 0) x0 += We;
  int x1 = x0 + 1; if (x1 == We) x1 = 0;
  const int y0 = min(max((int)s0, 0), He - 1), y1 = min(max((int)s0 + 1, 0), He - 1);
  // one 16-byte load per corner (the map is kept padded to RGBA): a query's four texels are four L1 requests instead of twelve --
  // the lanes of a warp look up unrelated texels, so every scalar load was up to 32 cache-line requests of its own
  const float4* r0 = e.env4 + (size_t)y0 * We;
  const float4* r1 = e.env4 + (size_t)y1 * We;
  const float4 e00 = __ldg(r0 + x0), e01 = __ldg(r0 + x1), e10 = __ldg(r1 + x0), e11 = __ldg(r1 + x1);
  float out[3];
  out[0] = (1.f - fs) * ((1.f - fu) * e00.x + fu * e01.x) + fs * ((1.f - fu) * e10.x + fu * e11.x);
  out[1] = (1.f - fs) * ((1.f - fu) * e00.y + fu * e01.y) + fs * ((1.f - fu) * e10.y + fu * e11.y);
  out[2] = (1.f - fs) * ((1.f - fu) * e00.z + fu * e01.z) + fs * ((1.f - fu) * e10.z + fu * e11.z);
  return make_float3(out[0], out[1], out[2]);
}

// ---- a10: f_r (n.w_i)^+ / p per channel (Q21-Q23) ---------------------------
__device__ __forceinline__ float sqrt_approx(float x) { float r; asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// The early return is kept on purpose.  (Measured and not kept: a branch-free version with a select at the end.  Secondary hits of
// neighbouring pixels have similar normals, so whole warps agree that a shared tertiary direction is back-facing and skip the
// specular term together: the branch-free kernel was slower, C3 16.7 -> 17.0 ms, C2 unchanged.)
__device__ __forceinline__ float3 brdf_cos_over_pdf(const ShadeP& sp, const float (&b)[7], float wix, float wiy, float wiz,
                                                    float wox, float woy, float woz, float pdf) {
  const float NoL = b[0] * wix + b[1] * wiy + b[2] * wiz;
  if (!(NoL > 0.f) || !(pdf > 0.f)) return make_float3(0.f, 0.f, 0.f);
  float spec = 0.f;
  if (sp.brdf_model == 1) {
    const float NoV = fmaxf(b[0] * wox + b[1] * woy + b[2] * woz, 1e-4f);
    float hx = wix + wox, hy = wiy + woy, hz = wiz + woz;
    const float hn = rsqrtf(fmaxf(hx * hx + hy * hy + hz * hz, 1e-24f));
    hx *= hn; hy *= hn; hz *= hn;
    const float NoH = fmaxf(b[0] * hx + b[1] * hy + b[2] * hz, 0.f);
    const float VoH = fmaxf(wox * hx + woy * hy + woz * hz, 0.f);
    const float alpha = b[6] * b[6], k = alpha * alpha;
    const float dd = NoH * NoH * (k - 1.f) + 1.f;
    const float m = 1.f - VoH, m2 = m * m;
    const float F = sp.f0 + (1.f - sp.f0) * (m2 * m2 * m);
    const float den = NoL * sqrt_approx(NoV * NoV * (1.f - k) + k) + NoV * sqrt_approx(NoL * NoL * (1.f - k) + k);
    spec = __fdividef(0.5f * k * F, 3.14159265358979f * dd * dd * den);        // D F G_v
  }
  const float sc = __fdividef(NoL, pdf);
  const float ipi = 0.3183098861837907f;
  return make_float3((b[3] * ipi + spec) * sc, (b[4] * ipi + spec) * sc, (b[5] * ipi + spec) * sc);
}

// incoming radiance for direction s of point-row i (Lin if supplied, else the env map)
__device__ __forceinline__ float3 incoming(const EnvP& e, const DirsetP& d, unsigned long long i, uint32_t s,
                                           float wx, float wy, float wz) {
  if (d.Lin) {
    const float* p = d.Lin + i * d.stride + 3ull * s;
    return make_float3(__ldg(p), __ldg(p + 1), __ldg(p + 2));
  }
  return env_lookup(e, wx, wy, wz);
}

}  // namespace hr
