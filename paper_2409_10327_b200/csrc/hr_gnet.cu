// hr_gnet.cu -- C-ABI entry points hashrender_gbuffer_* (include/hashrender.h): the CNN direct-illumination renderer G
// on tcgen05 + TMA.  Host side: weight re-layout, tensor maps, the launch sequence.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/hashrender.h"
#include "hr_gnet.cuh"

using namespace hr;
using namespace hr::gn;

namespace {

struct Layer {
  int Cout = 0, Cin = 0, k = 1;
  bool norm = true;
  int Kw = 0;                   // per-tap K extent of the fp16 weight tensor (multiple of 64)
  int kchunks = 0, wchunks = 0;
  __half* d_w = nullptr;        // [Cout][taps * Kw], K-major (conv layers)
  float* d_w32 = nullptr;       // [11][Cin] (map layers)
  float* d_b = nullptr; float* d_g = nullptr; float* d_be = nullptr;
  double* d_stats = nullptr;    // [2][Cout]
  CUtensorMap tmB;
  CUtensorMap tmA;
};

}  // namespace

struct hr_gnet {
  hr_gnet_config cfg;
  int num_sms = 148;
  std::vector<Layer> layers;    // stem, n_res residual layers, then per SR block: conv a, conv b, map
  // buffers
  __half* actIn = nullptr;      // [N0][64]
  __half* actF = nullptr;       // [N0][2 width]
  float* res = nullptr;         // [N0][width]
  float* pre = nullptr;         // largest [N][Cout]
  __half* actA[3] = {nullptr, nullptr, nullptr};
  __half* actB[3] = {nullptr, nullptr, nullptr};
  float* feat[3] = {nullptr, nullptr, nullptr};
  float* maps[3] = {nullptr, nullptr, nullptr};
  double* stats = nullptr; size_t stats_bytes = 0;
  std::vector<void*> owned;
  uint64_t launches = 0;
  double flops = 0;             // algorithmic flops of one forward (2 N Cout Cin taps per convolution, one pass)
  char err[512];
};

namespace {

int gfail(hr_gnet* h, int code, const char* fmt, ...) {
  if (h) {
    va_list ap; va_start(ap, fmt);
    vsnprintf(h->err, sizeof(h->err), fmt, ap);
    va_end(ap);
  }
  return code;
}
#define G_CUDA(h, call)                                                                                 \
  do {                                                                                                  \
    cudaError_t e_ = (call);                                                                            \
    if (e_ != cudaSuccess)                                                                              \
      return gfail(h, e_ == cudaErrorMemoryAllocation ? HR_ERR_OOM : HR_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); \
  } while (0)

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// fp16 tensor, innermost dimension first; 128-byte swizzle; out-of-bounds elements read as zero
bool make_map(CUtensorMap* tm, void* base, int rank, const uint64_t* dims, const uint32_t* box) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t gd[3]; cuuint64_t gs[2]; cuuint32_t bx[3]; cuuint32_t es[3] = {1, 1, 1};
  uint64_t stride = 2;
  for (int i = 0; i < rank; ++i) {
    gd[i] = dims[i]; bx[i] = box[i];
    stride *= dims[i];
    if (i < rank - 1) gs[i] = stride;
  }
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, rank, base, gd, gs, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <typename T>
int dev_alloc(hr_gnet* h, T** p, size_t n, bool zero) {
  G_CUDA(h, cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T)));
  h->owned.push_back(*p);
  if (zero) G_CUDA(h, cudaMemset(*p, 0, n * sizeof(T)));
  return HR_OK;
}
template <typename T>
int dev_upload(hr_gnet* h, T** p, const std::vector<T>& v) {
  if (int e = dev_alloc(h, p, v.size(), false)) return e;
  G_CUDA(h, cudaMemcpy(*p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
  return HR_OK;
}

int ew_grid(const hr_gnet* h, long long total, int nt) {
  long long need = (total + nt - 1) / nt, cap = (long long)h->num_sms * 8;
  return (int)(need < cap ? need : cap);
}

}  // namespace

extern "C" {

int hashrender_gbuffer_create(const hr_gnet_config* cfg, const float* weights, uint64_t n_weights, hr_gnet_t** out) {
  if (!out) return HR_ERR_INVALID_ARG;
  *out = nullptr;
  if (!cfg || !weights) return HR_ERR_INVALID_ARG;
  hr_gnet* h = new (std::nothrow) hr_gnet();
  if (!h) return HR_ERR_OOM;
  h->err[0] = 0;
  *out = h;
  h->cfg = *cfg;
  const int width = (int)cfg->width, n_res = (int)cfg->n_res;
  if (cfg->h < 1 || cfg->w < 1 || (uint64_t)cfg->h * cfg->w > (1u << 16)) return gfail(h, HR_ERR_INVALID_ARG, "gbuffer: ray array must hold 1 .. 65536 rays");
  if (width % 64 || width < 64 || width > 256 || n_res % 2 || n_res < 0 || n_res > 256)
    return gfail(h, HR_ERR_UNSUPPORTED, "gbuffer: need width in {64,128,192,256} and an even number of residual layers");
  for (int s = 0; s < 3; ++s)
    if (cfg->sr_ch[s] % 32 || cfg->sr_ch[s] < 32 || cfg->sr_ch[s] > 256 || (cfg->sr_ch[s] > 32 && cfg->sr_ch[s] % 64))
      return gfail(h, HR_ERR_UNSUPPORTED, "gbuffer: SR-block channels must be 32 or a multiple of 64 up to 256");
  if (!encode_fn()) return gfail(h, HR_ERR_CUDA, "gbuffer: cuTensorMapEncodeTiled is not available");
  int dev = 0;
  G_CUDA(h, cudaGetDevice(&dev));
  G_CUDA(h, cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev));
  G_CUDA(h, cudaFuncSetAttribute(k_gconv<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kConvSmem));
  G_CUDA(h, cudaFuncSetAttribute(k_gconv<9>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kConvSmem));

  // ---- layer table (blob order: stem, residual layers, then per SR block conv a, conv b, map) --------------------------------------
  std::vector<Layer>& L = h->layers;
  auto add = [&](int co, int ci, int k, bool norm) { Layer l; l.Cout = co; l.Cin = ci; l.k = k; l.norm = norm; L.push_back(l); };
  add(width, 6, 1, true);
  for (int i = 0; i < n_res; ++i) add(width, width, 1, true);
  int c = width;
  for (int s = 0; s < 3; ++s) { add(cfg->sr_ch[s], c, 3, true); add(cfg->sr_ch[s], cfg->sr_ch[s], 3, true); add(kOutCh, cfg->sr_ch[s], 1, false); c = cfg->sr_ch[s]; }
  uint64_t need = 0;
  for (const Layer& l : L) need += (uint64_t)l.Cout * l.Cin * l.k * l.k + l.Cout + (l.norm ? 2 * l.Cout : 0);
  if (need != n_weights) return gfail(h, HR_ERR_INVALID_ARG, "gbuffer: weight blob holds %llu floats, the architecture needs %llu",
                                      (unsigned long long)n_weights, (unsigned long long)need);
  size_t stats_n = 0;
  for (const Layer& l : L) if (l.norm) stats_n += 2 * l.Cout;
  if (int e = dev_alloc(h, &h->stats, stats_n, true)) return e;
  h->stats_bytes = stats_n * sizeof(double);

  // ---- weights ---------------------------------------------------------------------------------------------------------------------
  const float* p = weights;
  size_t stats_off = 0;
  for (Layer& l : L) {
    const int taps = l.k * l.k;
    const float* W = p; p += (size_t)l.Cout * l.Cin * taps;
    std::vector<float> b(p, p + l.Cout); p += l.Cout;
    if (int e = dev_upload(h, &l.d_b, b)) return e;
    if (!l.norm) {                                          // output-mapping layer: plain fp32 weights [11][Cin]
      std::vector<float> w(W, W + (size_t)l.Cout * l.Cin);
      if (int e = dev_upload(h, &l.d_w32, w)) return e;
      continue;
    }
    std::vector<float> g(p, p + l.Cout); p += l.Cout;
    std::vector<float> be(p, p + l.Cout); p += l.Cout;
    if (int e = dev_upload(h, &l.d_g, g)) return e;
    if (int e = dev_upload(h, &l.d_be, be)) return e;
    l.d_stats = h->stats + stats_off; stats_off += 2 * l.Cout;
    // activation K = [hi | lo].  Cin a multiple of 64: the lo chunks re-use the hi chunks' weights.  Cin < 64 (the 6-channel ray
    // input, 32 channels): hi and lo share ONE 64-channel chunk, so the weights are written twice inside it.
    const bool packed = l.Cin % 64 != 0;
    if (packed && 2 * l.Cin > 64) return gfail(h, HR_ERR_UNSUPPORTED, "gbuffer: %d input channels", l.Cin);
    l.Kw = packed ? 64 : l.Cin;
    l.wchunks = l.Kw / 64;
    l.kchunks = packed ? 1 : 2 * l.wchunks;
    std::vector<__half> wh((size_t)l.Cout * taps * l.Kw, __float2half_rn(0.f));
    for (int o = 0; o < l.Cout; ++o)
      for (int ci = 0; ci < l.Cin; ++ci)
        for (int t = 0; t < taps; ++t) {
          const float v = W[((size_t)o * l.Cin + ci) * taps + t];
          const __half hv = __float2half_rn(v);
          if (__half2float(hv) != v)
            return gfail(h, HR_ERR_INVALID_ARG, "gbuffer: convolution weights must be fp16-representable (layer with %d -> %d channels)", l.Cin, l.Cout);
          wh[((size_t)o * taps + t) * l.Kw + ci] = hv;
          if (packed) wh[((size_t)o * taps + t) * l.Kw + l.Cin + ci] = hv;
        }
    if (int e = dev_upload(h, &l.d_w, wh)) return e;
    const uint64_t dims[2] = {(uint64_t)taps * l.Kw, (uint64_t)l.Cout};
    const uint32_t box[2] = {64, (uint32_t)l.Cout};
    if (!make_map(&l.tmB, l.d_w, 2, dims, box)) return gfail(h, HR_ERR_CUDA, "gbuffer: weight tensor map");
  }

  // ---- activation buffers and their tensor maps ----------------------------------------------------------------------------------------
  const long long N0 = (long long)cfg->h * cfg->w;
  if (int e = dev_alloc(h, &h->actIn, (size_t)N0 * 64, true)) return e;
  if (int e = dev_alloc(h, &h->actF, (size_t)N0 * 2 * width, true)) return e;
  if (int e = dev_alloc(h, &h->res, (size_t)N0 * width, true)) return e;
  size_t pre_n = (size_t)N0 * width;
  int Hs = cfg->h, Ws = cfg->w;
  c = width;
  for (int s = 0; s < 3; ++s) {
    Hs *= 2; Ws *= 2;
    const int cs = cfg->sr_ch[s];
    const size_t Ns = (size_t)Hs * Ws, Np = (size_t)(Hs + 2) * (Ws + 2);
    pre_n = pre_n > Ns * cs ? pre_n : Ns * cs;
    if (int e = dev_alloc(h, &h->actA[s], Np * 2 * c, true)) return e;
    if (int e = dev_alloc(h, &h->actB[s], Np * 2 * cs, true)) return e;
    if (int e = dev_alloc(h, &h->feat[s], Ns * cs, false)) return e;
    if (int e = dev_alloc(h, &h->maps[s], Ns * kOutCh, false)) return e;
    c = cs;
  }
  if (int e = dev_alloc(h, &h->pre, pre_n, false)) return e;
  {
    const uint64_t d0[2] = {64, (uint64_t)N0}; const uint32_t b0[2] = {64, 128};
    if (!make_map(&L[0].tmA, h->actIn, 2, d0, b0)) return gfail(h, HR_ERR_CUDA, "gbuffer: tensor map");
    const uint64_t d1[2] = {(uint64_t)2 * width, (uint64_t)N0};
    for (int i = 1; i <= n_res; ++i)
      if (!make_map(&L[i].tmA, h->actF, 2, d1, b0)) return gfail(h, HR_ERR_CUDA, "gbuffer: tensor map");
    Hs = cfg->h; Ws = cfg->w; c = width;
    for (int s = 0; s < 3; ++s) {
      Hs *= 2; Ws *= 2;
      const int cs = cfg->sr_ch[s];
      const uint32_t b3[3] = {64, 8, 16};
      const uint64_t da[3] = {(uint64_t)2 * c, (uint64_t)Ws + 2, (uint64_t)Hs + 2}, db[3] = {(uint64_t)2 * cs, (uint64_t)Ws + 2, (uint64_t)Hs + 2};
      if (!make_map(&L[1 + n_res + 3 * s].tmA, h->actA[s], 3, da, b3) || !make_map(&L[2 + n_res + 3 * s].tmA, h->actB[s], 3, db, b3))
        return gfail(h, HR_ERR_CUDA, "gbuffer: tensor map");
      c = cs;
    }
  }
  // algorithmic work of one forward
  h->flops = 0;
  {
    double n = (double)N0;
    for (int i = 0; i <= n_res; ++i) h->flops += 2.0 * n * L[i].Cout * L[i].Cin;
    for (int s = 0; s < 3; ++s) {
      n *= 4;
      for (int j = 0; j < 3; ++j) { const Layer& l = L[1 + n_res + 3 * s + j]; h->flops += 2.0 * n * l.Cout * l.Cin * l.k * l.k; }
    }
  }
  return HR_OK;
}

int hashrender_gbuffer_destroy(hr_gnet_t* h) {
  if (!h) return HR_ERR_INVALID_ARG;
  cudaDeviceSynchronize();
  for (void* p : h->owned) cudaFree(p);
  delete h;
  return HR_OK;
}

static int launch_conv(hr_gnet* h, const Layer& l, int H, int W, cudaStream_t st) {
  ConvP p;
  p.taps = l.k * l.k; p.kchunks = l.kchunks; p.wchunks = l.wchunks; p.Cout = l.Cout; p.H = H; p.W = W; p.N = (long long)H * W;
  p.bias = l.d_b; p.pre = h->pre; p.stats = l.d_stats;
  if (l.k == 3) { p.tiles_x = (W + 7) / 8; p.tiles = p.tiles_x * ((H + 15) / 16); }
  else { p.tiles_x = 1; p.tiles = (int)((p.N + 127) / 128); }
  const int grid = p.tiles < h->num_sms ? p.tiles : h->num_sms;
  if (l.k == 3) k_gconv<9><<<grid, 192, kConvSmem, st>>>(l.tmA, l.tmB, p);
  else k_gconv<1><<<grid, 192, kConvSmem, st>>>(l.tmA, l.tmB, p);
  h->launches++;
  G_CUDA(h, cudaGetLastError());
  return HR_OK;
}
static int launch_norm(hr_gnet* h, const Layer& l, int H, int W, int mode, float* res, float* feat, __half* act, cudaStream_t st) {
  NormP p;
  p.pre = h->pre; p.stats = l.d_stats; p.gamma = l.d_g; p.beta = l.d_be; p.res = res; p.feat = feat; p.act = act;
  p.N = (long long)H * W; p.C = l.Cout; p.H = H; p.W = W; p.mode = mode;
  k_gnorm<<<ew_grid(h, p.N * (p.C / 8), 256), 256, 2 * p.C * sizeof(float), st>>>(p);
  h->launches++;
  G_CUDA(h, cudaGetLastError());
  return HR_OK;
}

int hashrender_gbuffer_forward(hr_gnet_t* h, const float* rays, float* x, float* brdf, uint8_t* mask, float* raw, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (!rays || (!x && !brdf && !mask && !raw)) return gfail(h, HR_ERR_INVALID_ARG, "gbuffer_forward: NULL rays or no output requested");
  cudaStream_t st = (cudaStream_t)stream;
  const hr_gnet_config& cfg = h->cfg;
  const int n_res = (int)cfg.n_res;
  std::vector<Layer>& L = h->layers;
  const long long N0 = (long long)cfg.h * cfg.w;
  G_CUDA(h, cudaMemsetAsync(h->stats, 0, h->stats_bytes, st));
  k_grays<<<ew_grid(h, N0 * 6, 256), 256, 0, st>>>(rays, h->actIn, N0);
  h->launches++;
  // stem + residual MLP: 1x1 conv-norm-act layers on the flat pixel matrix
  if (int e = launch_conv(h, L[0], cfg.h, cfg.w, st)) return e;
  if (int e = launch_norm(h, L[0], cfg.h, cfg.w, 0, h->res, nullptr, h->actF, st)) return e;
  for (int i = 1; i <= n_res; ++i) {
    if (int e = launch_conv(h, L[i], cfg.h, cfg.w, st)) return e;
    if (int e = launch_norm(h, L[i], cfg.h, cfg.w, (i & 1) ? 1 : 2, h->res, nullptr, h->actF, st)) return e;
  }
  // three SR blocks (PAPER.md:68b) with the output skip (PAPER.md:68a)
  int Hs = cfg.h, Ws = cfg.w, c = (int)cfg.width;
  const float* src = h->res;
  for (int s = 0; s < 3; ++s) {
    k_gupsample<<<ew_grid(h, (long long)4 * Hs * Ws * (c / 8), 256), 256, 0, st>>>(src, h->actA[s], Hs, Ws, c);
    h->launches++;
    Hs *= 2; Ws *= 2;
    const Layer& la = L[1 + n_res + 3 * s]; const Layer& lb = L[2 + n_res + 3 * s]; const Layer& lm = L[3 + n_res + 3 * s];
    if (int e = launch_conv(h, la, Hs, Ws, st)) return e;
    if (int e = launch_norm(h, la, Hs, Ws, 4, nullptr, nullptr, h->actB[s], st)) return e;
    if (int e = launch_conv(h, lb, Hs, Ws, st)) return e;
    if (int e = launch_norm(h, lb, Hs, Ws, 3, nullptr, h->feat[s], nullptr, st)) return e;
    MapP m;
    m.feat = h->feat[s]; m.Wm = lm.d_w32; m.bm = lm.d_b; m.prev = s ? h->maps[s - 1] : nullptr; m.H = Hs; m.W = Ws; m.C = lm.Cin;
    const bool last = s == 2;
    m.out = last ? raw : h->maps[s];
    m.x = last ? x : nullptr; m.brdf = last ? brdf : nullptr; m.mask = last ? mask : nullptr; m.rough_min = cfg.rough_min;
    k_gmap<<<ew_grid(h, (long long)Hs * Ws, 128), 128, (kOutCh * m.C + kOutCh) * sizeof(float), st>>>(m);
    h->launches++;
    src = h->feat[s];
    c = lm.Cin;
  }
  G_CUDA(h, cudaGetLastError());
  return HR_OK;
}

uint64_t hashrender_gbuffer_launch_count(const hr_gnet_t* h) { return h ? h->launches : 0; }
double hashrender_gbuffer_flops(const hr_gnet_t* h) { return h ? h->flops : 0.0; }
const char* hashrender_gbuffer_last_error(const hr_gnet_t* h) { return h ? h->err : "NULL handle"; }

}  // extern "C"
