// hashrender.cu -- C-ABI entry points (include/hashrender.h) and host-side launch logic.
// Argument validation happens before any launch; every kernel is enqueued on the caller's stream.
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/hashrender.h"
#include "hr_kernels_ffma.cuh"
#include "hr_kernels_tc.cuh"
#include "hr_sampler.cuh"
#include "hr_svgf.cuh"
#include "hr_wg_api.h"

using namespace hr;

struct hashrender {
  hr_config cfg;
  uint32_t res[kMaxL];
  GridP grid;
  ShadeP shade;
  EnvP env;
  void* d_tables = nullptr;
  uint64_t table_bytes = 0;      // size of the device copy of the tables (all layouts)
  float* d_wts = nullptr;        // prepared fp32 weights (hr_kernels_ffma.cuh layout)
  uint8_t* d_wts_tc = nullptr;   // fp16 UMMA weight tiles, hi then lo halves (hr_render_wg.cuh)
  std::vector<uint8_t> h_wts_tc; // host copy of [TcConst | hi tiles | lo tiles]; TcConst is passed by value at launch
  void* d_ring = nullptr;        // work-item rings of the render kernel (one per warpgroup)
  unsigned long long* d_counters = nullptr;   // [0] tile counter, [1] items evaluated, [2] secondary rays traced
  bool split_ok = false;         // fp32 model representable as fp16 hi + lo without overflow (enables the tcgen05 fp32 path)
  float* d_env = nullptr;
  float4* d_env4 = nullptr;      // the env map padded to RGBA
  size_t env_cap = 0;
  int num_sms = 148;
  uint64_t launches = 0;
  const char* last_path = "none";
  char err[512];
  // staging for render_frame_host
  void* stage[16] = {nullptr};
  size_t stage_cap[16] = {0};
  void* d_svgf = nullptr;        // denoiser scratch: geo | live | two colour+variance planes
  size_t svgf_cap = 0;
  float* d_light = nullptr;      // sampler tables: pmf [He*We] then cdf [He*We] (built lazily from the env map)
  size_t light_cap = 0;
  bool light_valid = false;
  cudaStream_t copy_stream = nullptr;   // render_frame_host: H2D copies of chunk c+1 overlap the render of chunk c
  cudaEvent_t ev[9] = {nullptr};
};

namespace {

int fail(hashrender* h, int code, const char* fmt, ...) {
  if (h) {
    va_list ap; va_start(ap, fmt);
    vsnprintf(h->err, sizeof(h->err), fmt, ap);
    va_end(ap);
  }
  return code;
}

#define HR_CUDA(h, call)                                                                              \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess)                                                                            \
      return fail(h, e_ == cudaErrorMemoryAllocation ? HR_ERR_OOM : HR_ERR_CUDA, "%s failed: %s", #call, \
                  cudaGetErrorString(e_));                                                            \
  } while (0)

__global__ void k_env_pack(const float* __restrict__ src, float4* __restrict__ dst, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    dst[i] = make_float4(src[3 * i], src[3 * i + 1], src[3 * i + 2], 0.f);
}

__global__ void k_f32_to_f16(const float* __restrict__ src, __half* __restrict__ dst, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    dst[i] = __float2half_rn(src[i]);
}

// Cell-major copy of one level (hr_device.cuh GridP): entry e = cx + N (cy + N cz) <- the 8 corner rows, each read at the SPECIFIED
// index (corner_indices: dense x + y (N+1) + z (N+1)^2, or the hash) from the caller's rows `src` of that level.
template <bool F16>
__global__ void k_build_cells(const float2* __restrict__ src, uint32_t N, bool dense, uint32_t log2_T, void* __restrict__ dst) {
  const size_t cells = (size_t)N * N * N;
  for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < cells; e += (size_t)gridDim.x * blockDim.x) {
    Cell c;
    c.c0[0] = (uint32_t)(e % N); c.c0[1] = (uint32_t)((e / N) % N); c.c0[2] = (uint32_t)(e / ((size_t)N * N));
    uint32_t idx[8];
    corner_indices(c, N, dense, log2_T, idx);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float2 v = src[idx[k]];
      if (F16) reinterpret_cast<__half2*>(dst)[e * 8 + k] = __floats2half2_rn(v.x, v.y);
      else reinterpret_cast<float2*>(dst)[e * 8 + k] = v;
    }
  }
}

constexpr int NT_FFMA = 256;

void prepare_weights_ffma(const hr_config& c, const float* bw, const float* iw, std::vector<float>& out) {
  const int D = c.L * c.F, H = kH;
  out.assign(wo_::ALL, 0.f);
  float* B = out.data();
  float* I = out.data() + wo_::B_SIZE;
  {  // B: W1[H][D], b1[H], W2[H][H], b2[H], W3[7][H], b3[7]
    const float* W1 = bw; const float* b1 = W1 + H * D; const float* W2 = b1 + H; const float* b2 = W2 + H * H;
    const float* W3 = b2 + H; const float* b3 = W3 + 7 * H;
    for (int j = 0; j < H; ++j) for (int k = 0; k < D; ++k) B[wo_::B_W1 + k * H + j] = W1[j * D + k];
    for (int j = 0; j < H; ++j) B[wo_::B_b1 + j] = b1[j];
    for (int j = 0; j < H; ++j) for (int k = 0; k < H; ++k) B[wo_::B_W2 + k * H + j] = W2[j * H + k];
    for (int j = 0; j < H; ++j) B[wo_::B_b2 + j] = b2[j];
    for (int cidx = 0; cidx < 7; ++cidx) for (int k = 0; k < H; ++k) B[wo_::B_W3 + k * 8 + cidx] = W3[cidx * H + k];
    for (int cidx = 0; cidx < 7; ++cidx) B[wo_::B_b3 + cidx] = b3[cidx];
  }
  {  // I: W1[H][D+3], b1[H], W2[H][H], b2[H], W3[2][H], b3[2]
    const int Din = D + 3;
    const float* W1 = iw; const float* b1 = W1 + H * Din; const float* W2 = b1 + H; const float* b2 = W2 + H * H;
    const float* W3 = b2 + H; const float* b3 = W3 + 2 * H;
    for (int j = 0; j < H; ++j) for (int k = 0; k < D; ++k) I[wo_::I_W1f + k * H + j] = W1[j * Din + k];
    for (int j = 0; j < H; ++j) for (int d = 0; d < 3; ++d) I[wo_::I_W1w + d * H + j] = W1[j * Din + D + d];
    for (int j = 0; j < H; ++j) I[wo_::I_b1 + j] = b1[j];
    for (int j = 0; j < H; ++j) for (int k = 0; k < H; ++k) I[wo_::I_W2 + k * H + j] = W2[j * H + k];
    for (int j = 0; j < H; ++j) I[wo_::I_b2 + j] = b2[j];
    for (int cidx = 0; cidx < 2; ++cidx) for (int k = 0; k < H; ++k) I[wo_::I_W3 + k * 2 + cidx] = W3[cidx * H + k];
    for (int cidx = 0; cidx < 2; ++cidx) I[wo_::I_b3 + cidx] = b3[cidx];
  }
}

DirsetP to_dev(const hr_dirset& d) {
  DirsetP p; p.dir = d.dir; p.pdf = d.pdf; p.Lin = d.Lin; p.S = d.S; p.stride = d.point_stride; return p;
}

int grid_for(const hashrender* h, uint64_t N, int nt, int blocks_per_sm) {
  uint64_t need = (N + nt - 1) / nt;
  uint64_t cap = (uint64_t)h->num_sms * blocks_per_sm;
  return (int)(need < cap ? need : cap);
}

int check_dirset(hashrender* h, const hr_dirset* d, const char* name, bool need_pdf) {
  if (!d) return fail(h, HR_ERR_INVALID_ARG, "%s: NULL direction set", name);
  if (d->S == 0) return fail(h, HR_ERR_INVALID_ARG, "%s: S == 0", name);
  if (!d->dir) return fail(h, HR_ERR_INVALID_ARG, "%s: NULL dir", name);
  if (need_pdf && !d->pdf) return fail(h, HR_ERR_INVALID_ARG, "%s: NULL pdf", name);
  if (d->point_stride % 3 != 0) return fail(h, HR_ERR_INVALID_ARG, "%s: point_stride must be a multiple of 3", name);
  if (d->point_stride && d->point_stride < 3ull * d->S) return fail(h, HR_ERR_INVALID_ARG, "%s: point_stride < 3*S", name);
  return HR_OK;
}

// 0 = fp32 FFMA kernels, 1 = tcgen05 with fp16 activations, 2 = tcgen05 in hi/lo split precision (fp32 models)
int render_path(const hashrender* h) {
  if (!h->d_wts_tc) return 0;
  if (h->cfg.mlp_dtype == HR_F16) return 1;
  return h->split_ok ? 2 : 0;
}

// Upper bound of every hidden activation of an MLP whose inputs are bounded by in_max: the split-precision path holds
// activations as fp16 hi + lo, so they must stay far below 65504.
float mlp_bound(const float* w, int din, int H, float in_max) {
  const float* W1 = w; const float* b1 = W1 + H * din; const float* W2 = b1 + H; const float* b2 = W2 + H * H;
  float B1 = 0.f, B2 = 0.f;
  for (int j = 0; j < H; ++j) {
    float s = fabsf(b1[j]);
    for (int k = 0; k < din; ++k) s += fabsf(W1[j * din + k]) * in_max;
    B1 = fmaxf(B1, s);
  }
  for (int j = 0; j < H; ++j) {
    float s = fabsf(b2[j]);
    for (int k = 0; k < H; ++k) s += fabsf(W2[j * H + k]) * B1;
    B2 = fmaxf(B2, s);
  }
  return fmaxf(B1, B2);
}

// ---- hashrender_probe_gather: the rate at which an SM's L1 serves fully divergent loads (the roofline of the encode) -----------
// Every thread draws pseudo-random slots of a table and loads `group` consecutive W-byte words of each (group = 1: every load its own
// 32-byte sector; 2 / 4 / 8: that many loads per sector, as the corner rows of an x-pair are), eight independent slots in flight.
__device__ __forceinline__ uint32_t probe_mix(uint32_t x) { x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16; return x; }
template <int W> __device__ __forceinline__ uint32_t probe_ld(const uint8_t* p);
template <> __device__ __forceinline__ uint32_t probe_ld<4>(const uint8_t* p) { uint32_t v; asm volatile("ld.global.nc.b32 %0, [%1];" : "=r"(v) : "l"(p)); return v; }
template <> __device__ __forceinline__ uint32_t probe_ld<8>(const uint8_t* p) {
  uint32_t a, b; asm volatile("ld.global.nc.v2.b32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "l"(p)); return a ^ b;
}
template <> __device__ __forceinline__ uint32_t probe_ld<32>(const uint8_t* p) {
  uint32_t r[8];
  asm volatile("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "l"(p));
  return r[0] ^ r[1] ^ r[2] ^ r[3] ^ r[4] ^ r[5] ^ r[6] ^ r[7];
}
template <int W, int GROUP>
__global__ void k_probe_gather(const uint8_t* __restrict__ tab, uint32_t mask, int iters, uint32_t* sink, unsigned long long* cycles) {
  constexpr int IF = 8;                                               // independent slots in flight per thread
  uint32_t s = probe_mix(blockIdx.x * blockDim.x + threadIdx.x + 1u), acc = 0;
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
    uint32_t v[IF * GROUP];
#pragma unroll
    for (int q = 0; q < IF; ++q) {
      s = probe_mix(s + q + 1u);
#pragma unroll
      for (int e = 0; e < GROUP; ++e) v[q * GROUP + e] = probe_ld<W>(tab + (size_t)(((s & mask) & ~(uint32_t)(GROUP - 1)) + e) * W);
    }
#pragma unroll
    for (int q = 0; q < IF * GROUP; ++q) acc += v[q];
  }
  const long long t1 = clock64();
  if (acc == 0x12345u) sink[0] = acc;
  if (threadIdx.x == 0) atomicAdd(cycles, (unsigned long long)(t1 - t0));
}
template <int W, int GROUP>
cudaError_t run_probe(const uint8_t* tab, uint64_t bytes, int smem, int sms, uint32_t* sink, unsigned long long* cyc, double* per_cycle, double* per_s) {
  const uint32_t mask = (uint32_t)(bytes / W - 1);
  const int threads = 512, iters = 2048 / GROUP;
  cudaError_t e = cudaFuncSetAttribute(k_probe_gather<W, GROUP>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return e;
  k_probe_gather<W, GROUP><<<sms, threads, smem>>>(tab, mask, 16, sink, cyc);           // warm-up
  cudaMemset(cyc, 0, 8);
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  cudaEventRecord(a);
  k_probe_gather<W, GROUP><<<sms, threads, smem>>>(tab, mask, iters, sink, cyc);
  cudaEventRecord(b);
  e = cudaEventSynchronize(b);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, a, b);
  cudaEventDestroy(a); cudaEventDestroy(b);
  if (e != cudaSuccess) return e;
  unsigned long long c = 0;
  e = cudaMemcpy(&c, cyc, 8, cudaMemcpyDeviceToHost);
  const double loads = (double)threads * iters * 8 * GROUP;
  *per_cycle = loads / ((double)c / sms);
  *per_s = loads * sms / (ms * 1e-3);
  return e;
}

// ---- hashrender_denoise_static: the denoiser's image planes in a file-scope device array (no allocation, ever) ----------------
// Layout for an n-pixel image (n <= HASHRENDER_DENOISE_STATIC_MAX_PIXELS), the same as the handle-owned scratch of hashrender_denoise:
// geo [n] | live [n, padded to 16] | colour+variance plane A [n] | plane B [n].  Every GPU that loads the library holds the array until
// the process exits.  Pass 0 (k_svgf_prep) writes every byte the later passes read, so nothing here has to start at zero and the
// previous call's contents never show through.
constexpr size_t kSvgfStaticPixels = HASHRENDER_DENOISE_STATIC_MAX_PIXELS;
constexpr size_t kSvgfStaticBytes = kSvgfStaticPixels * (sizeof(svgf::Geo) + 2 * sizeof(float4)) + (kSvgfStaticPixels + 15) / 16 * 16;
static __device__ __align__(256) unsigned char g_svgf_static[kSvgfStaticBytes];

// In host code `g_svgf_static` is only the host-side stand-in of the symbol: the device address comes from cudaGetSymbolAddress,
// asked once per device with that device current (hashrender_create does, so the first denoise_static call finds it cached).
constexpr int kMaxDevices = 64;
char* g_svgf_static_base[kMaxDevices] = {nullptr};
cudaError_t g_svgf_static_err[kMaxDevices] = {cudaSuccess};
bool g_svgf_static_asked[kMaxDevices] = {false};
std::mutex g_svgf_static_mu;

cudaError_t svgf_static_base(char** base) {
  *base = nullptr;
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_svgf_static_mu);
  if (!g_svgf_static_asked[dev]) {
    void* p = nullptr;
    g_svgf_static_err[dev] = cudaGetSymbolAddress(&p, g_svgf_static);
    g_svgf_static_base[dev] = g_svgf_static_err[dev] == cudaSuccess ? static_cast<char*>(p) : nullptr;
    g_svgf_static_asked[dev] = g_svgf_static_err[dev] == cudaSuccess;     // a failed query is asked again on the next call
  }
  *base = g_svgf_static_base[dev];
  return g_svgf_static_err[dev];
}

}  // namespace

extern "C" {

int hashrender_create(const hr_config* cfg, const float* tables, const float* brdf_w, const float* irt_w, hashrender_t** out) {
  if (!out) return HR_ERR_INVALID_ARG;
  *out = nullptr;
  if (!cfg || !tables || !brdf_w || !irt_w || !cfg->res) return HR_ERR_INVALID_ARG;
  hashrender* h = new (std::nothrow) hashrender();
  if (!h) return HR_ERR_OOM;
  h->err[0] = 0;
  *out = h;   // returned even on failure so the caller can read last_error, then destroy
  h->cfg = *cfg;
  if (cfg->F != 2 || cfg->L < 1 || cfg->L > kMaxL || cfg->log2_T < 1 || cfg->log2_T > 28 || cfg->hidden != kH ||
      cfg->brdf_out != 7 || cfg->irt_out != 2)
    return fail(h, HR_ERR_UNSUPPORTED, "unsupported shape: need F==2, 1<=L<=16, 1<=log2_T<=28, hidden==64, brdf_out==7, irt_out==2");
  if (cfg->table_dtype > 1 || cfg->mlp_dtype > 1 || cfg->vis_mode > 1 || cfg->brdf_model > 1)
    return fail(h, HR_ERR_INVALID_ARG, "bad dtype / mode enum");
  for (uint32_t l = 0; l < cfg->L; ++l) {
    h->res[l] = cfg->res[l];
    if (cfg->res[l] < 1 || cfg->res[l] > (1u << 24)) return fail(h, HR_ERR_INVALID_ARG, "res[%u] out of range", l);
  }
  h->cfg.res = h->res;
  int dev = 0;
  HR_CUDA(h, cudaGetDevice(&dev));
  HR_CUDA(h, cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev));

  // grid parameters + the device layout of the tables (hr_device.cuh GridP): hashed levels keep their T rows; a dense level is stored
  // with power-of-two strides (row = cx | cy << b | cz << 2b), so one XOR index path serves every level
  GridP& g = h->grid;
  g.L = cfg->L; g.log2_T = cfg->log2_T; g.f16 = cfg->table_dtype; g.dense_mask = 0;
  const uint64_t T = 1ull << cfg->log2_T;
  const size_t esz = cfg->table_dtype == HR_F32 ? 8 : 4;               // bytes per row (F = 2)
  uint64_t rows_total = 0, lvl_rows[kMaxL], lvl_bits[kMaxL];
  for (uint32_t l = 0; l < kMaxL; ++l) { g.res[l] = 1; g.pa[l] = g.pb[l] = g.pmask[l] = 0; g.off[l] = 0; lvl_rows[l] = 0; lvl_bits[l] = 0; }
  // Cell-major levels: the coarsest levels whose 8-rows-per-cell copies fit a byte budget.  Tables that fit the L2 keep the copies
  // to a quarter of it, so that the working set stays resident; larger tables stream from HBM anyway and get four times their own
  // size.  Measured with k_trace_wg, 2^24 points, fp16 (ms without -> with): T = 2^19 6.25 -> 4.95 (27 MB of copies; 71 MB: 5.13),
  // 2^20 6.26 -> 5.64 (71 MB: 6.25), 2^21 9.67 -> 7.82 (491 MB), 2^22 11.93 -> 8.83 (491 MB; 1.3 GB: 8.36), 2^24 12.76 -> 9.52
  // (3.4 GB; 1.3 GB: 10.28, 9.1 GB: 8.86).
  g.nblock = 0;
  {
    int l2 = 0;
    HR_CUDA(h, cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev));
    const uint64_t table_bytes = ((uint64_t)cfg->L << cfg->log2_T) * esz;
    uint64_t budget = table_bytes <= (uint64_t)l2 ? (uint64_t)l2 / 4 : 4 * table_bytes;
    size_t mem_free = 0, mem_total = 0;
    HR_CUDA(h, cudaMemGetInfo(&mem_free, &mem_total));
    if (budget > mem_free / 4) budget = mem_free / 4;                 // the copies are an optimisation: never crowd out the caller
    if (cfg->log2_T > 26) budget = 0;                                 // the build stages one level's rows (T x 8 bytes) on the device
    uint64_t cum = 0;
    for (uint32_t l = 0; l < cfg->L; ++l) {
      const uint64_t N = cfg->res[l], b = N * N * N * 8 * esz;
      if (N * N * N > (1ull << 28) || cum + b > budget) break;
      cum += b; g.nblock = l + 1;
    }
  }
  for (uint32_t l = 0; l < cfg->L; ++l) {
    g.res[l] = cfg->res[l];
    const uint64_t sN = (uint64_t)cfg->res[l] + 1;
    if (l < g.nblock) {                                               // 8 rows per cell; entries stay sector-aligned (block levels come first)
      if (sN * sN * sN <= T) g.dense_mask |= 1u << l;
      lvl_rows[l] = (uint64_t)cfg->res[l] * cfg->res[l] * cfg->res[l] * 8;
    } else if (sN * sN * sN <= T) {
      g.dense_mask |= 1u << l;
      uint32_t bx = 1;
      while ((1ull << bx) < sN) ++bx;
      lvl_bits[l] = bx;
      g.pa[l] = 1u << bx; g.pb[l] = 1u << (2 * bx); g.pmask[l] = 0xFFFFFFFFu;
      lvl_rows[l] = sN << (2 * bx);                                   // z-slabs 0 .. N
    } else {
      g.pa[l] = 2654435761u; g.pb[l] = 805459861u; g.pmask[l] = (uint32_t)(T - 1);
      lvl_rows[l] = T;
    }
    g.off[l] = rows_total * esz;
    rows_total += (lvl_rows[l] + 3) & ~3ull;                          // keep every level 16-byte aligned
  }
  const uint64_t zero_off = rows_total * esz;
  rows_total += 8;                                                    // zero rows for the null levels l >= L
  for (uint32_t l = cfg->L; l < kMaxL; ++l) g.off[l] = zero_off;
  {
    int l2 = 0;
    HR_CUDA(h, cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev));
    uint64_t hashed = 0;
    for (uint32_t l = g.nblock; l < cfg->L; ++l) if (!((g.dense_mask >> l) & 1u)) hashed += lvl_rows[l] * esz;
    g.l2_hint = hashed > 2ull * (uint64_t)l2 ? 1u : 0u;                // measured: helps at 448 MB of hashed levels, hurts at 128 MB (hr_device.cuh)
  }
  {
    int l2 = 0;
    HR_CUDA(h, cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev));
    g.pair_loads = (cfg->table_dtype == HR_F16 && rows_total * esz <= (uint64_t)l2 / 2) ? 1u : 0u;   // L2-resident on both dies' halves
  }
  HR_CUDA(h, cudaMalloc(&h->d_tables, rows_total * esz));
  h->table_bytes = rows_total * esz;
  HR_CUDA(h, cudaMemset(h->d_tables, 0, rows_total * esz));
  const size_t n = (size_t)cfg->L << cfg->log2_T << 1;                  // floats in the caller's [L][T][2] array
  {
    const size_t chunk = (size_t)16 << 20;                            // floats per staged piece (fp16 tables are converted on the device)
    float* st = nullptr;
    if (cfg->table_dtype == HR_F16) HR_CUDA(h, cudaMalloc(&st, chunk * sizeof(float)));
    std::vector<float> relaid;
    cudaError_t e = cudaSuccess;
    float2* lvl_src = nullptr;                                        // one level's rows as given, for the cell-major build
    if (g.nblock) e = cudaMalloc(&lvl_src, (size_t)T * sizeof(float2));
    for (uint32_t l = 0; l < g.nblock && e == cudaSuccess; ++l) {
      const uint64_t sN = (uint64_t)cfg->res[l] + 1;
      const bool dense = (g.dense_mask >> l) & 1u;
      e = cudaMemcpy(lvl_src, tables + ((size_t)l << cfg->log2_T) * 2, (dense ? sN * sN * sN : T) * sizeof(float2), cudaMemcpyHostToDevice);
      if (e != cudaSuccess) break;
      void* dst = reinterpret_cast<char*>(h->d_tables) + g.off[l];
      if (cfg->table_dtype == HR_F16) k_build_cells<true><<<h->num_sms * 8, 256>>>(lvl_src, cfg->res[l], dense, cfg->log2_T, dst);
      else k_build_cells<false><<<h->num_sms * 8, 256>>>(lvl_src, cfg->res[l], dense, cfg->log2_T, dst);
      e = cudaDeviceSynchronize();
    }
    cudaFree(lvl_src);
    for (uint32_t l = g.nblock; l < cfg->L && e == cudaSuccess; ++l) {
      const float* src = tables + ((size_t)l << cfg->log2_T) * 2;
      if ((g.dense_mask >> l) & 1u) {                                 // vertex (x, y, z): row x + y s + z s^2 -> row x | y << b | z << 2b
        const uint64_t sN = (uint64_t)cfg->res[l] + 1, bx = lvl_bits[l];
        relaid.assign(lvl_rows[l] * 2, 0.f);
        for (uint64_t z = 0; z < sN; ++z)
          for (uint64_t y = 0; y < sN; ++y)
            memcpy(&relaid[((z << (2 * bx)) | (y << bx)) * 2], src + (y * sN + z * sN * sN) * 2, sN * 2 * sizeof(float));
        src = relaid.data();
      }
      const size_t nf = lvl_rows[l] * 2;
      char* dst = reinterpret_cast<char*>(h->d_tables) + g.off[l];
      if (cfg->table_dtype == HR_F32) {
        e = cudaMemcpy(dst, src, nf * sizeof(float), cudaMemcpyHostToDevice);
      } else {
        for (size_t o = 0; o < nf && e == cudaSuccess; o += chunk) {
          const size_t m = nf - o < chunk ? nf - o : chunk;
          e = cudaMemcpy(st, src + o, m * sizeof(float), cudaMemcpyHostToDevice);
          if (e == cudaSuccess) {
            k_f32_to_f16<<<h->num_sms * 8, 256>>>(st, reinterpret_cast<__half*>(dst) + o, m);
            e = cudaDeviceSynchronize();
          }
        }
      }
    }
    cudaFree(st);
    if (e != cudaSuccess) return fail(h, HR_ERR_CUDA, "table upload failed: %s", cudaGetErrorString(e));
  }
  g.tables = h->d_tables;
  // weights
  std::vector<float> w;
  prepare_weights_ffma(*cfg, brdf_w, irt_w, w);
  HR_CUDA(h, cudaMalloc(&h->d_wts, w.size() * sizeof(float)));
  HR_CUDA(h, cudaMemcpy(h->d_wts, w.data(), w.size() * sizeof(float), cudaMemcpyHostToDevice));
  {
    size_t cb = 0, tb = 0;
    wg::prepare_weights_blob(*cfg, brdf_w, irt_w, h->h_wts_tc, &cb, &tb);
    HR_CUDA(h, cudaMalloc(&h->d_wts_tc, tb));
    HR_CUDA(h, cudaMemcpy(h->d_wts_tc, h->h_wts_tc.data() + cb, tb, cudaMemcpyHostToDevice));
    HR_CUDA(h, cudaMalloc(&h->d_ring, wg::ring_bytes(h->num_sms)));
    HR_CUDA(h, cudaMalloc(&h->d_counters, 4 * sizeof(unsigned long long)));
    HR_CUDA(h, cudaMemset(h->d_counters, 0, 4 * sizeof(unsigned long long)));
    // fp32 model on the fp16 tensor cores: every value is carried as fp16 hi + lo, so tables, weights and hidden
    // activations must be finite and well inside the fp16 range
    float tmax = 0.f;
    for (size_t i = 0; i < n; ++i) tmax = fmaxf(tmax, fabsf(tables[i]));
    const int D = cfg->L * cfg->F;
    const float fb = fmaxf(tmax, 1.f);
    const float bound = fmaxf(mlp_bound(brdf_w, D, kH, fb), mlp_bound(irt_w, D + 3, kH, fb));
    h->split_ok = tmax < 1024.f && bound < 16384.f;      // NaN fails both comparisons
  }
  ShadeP& s = h->shade;
  s.near_t = cfg->near_t; s.far_t = cfg->far_t; s.rough_min = cfg->rough_min; s.f0 = cfg->fresnel_f0;
  s.vis_mode = cfg->vis_mode; s.brdf_model = cfg->brdf_model;
  s.as0 = cfg->albedo_scale[0]; s.as1 = cfg->albedo_scale[1]; s.as2 = cfg->albedo_scale[2];
  h->env.env = nullptr; h->env.env4 = nullptr; h->env.He = h->env.We = 0;

  const int smem_full = (int)ffma_smem_bytes(NT_FFMA, true), smem_half = (int)ffma_smem_bytes(NT_FFMA, false);
  HR_CUDA(h, cudaFuncSetAttribute(k_render_ffma<false, NT_FFMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_full));
  HR_CUDA(h, cudaFuncSetAttribute(k_render_ffma<true, NT_FFMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_full));
  HR_CUDA(h, cudaFuncSetAttribute(k_trace_ffma<false, NT_FFMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_half));
  HR_CUDA(h, cudaFuncSetAttribute(k_trace_ffma<true, NT_FFMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_half));
  HR_CUDA(h, cudaFuncSetAttribute(k_decode_ffma<NT_FFMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_half));
  HR_CUDA(h, wg::init_device_p0());      // per device (a second handle on another device opts in there too)
  HR_CUDA(h, wg::init_device_p1());
  { char* b = nullptr; (void)svgf_static_base(&b); }   // set-up for hashrender_denoise_static; a failure is reported by that call
  return HR_OK;
}

int hashrender_destroy(hashrender_t* h) {
  if (!h) return HR_ERR_INVALID_ARG;
  cudaDeviceSynchronize();
  cudaFree(h->d_tables); cudaFree(h->d_wts); cudaFree(h->d_wts_tc); cudaFree(h->d_env); cudaFree(h->d_env4);
  cudaFree(h->d_ring); cudaFree(h->d_counters); cudaFree(h->d_light); cudaFree(h->d_svgf);
  if (h->copy_stream) {
    cudaStreamDestroy(h->copy_stream);
    for (int i = 0; i < 9; ++i) cudaEventDestroy(h->ev[i]);
  }
  for (int i = 0; i < 16; ++i) cudaFree(h->stage[i]);
  delete h;
  return HR_OK;
}

int hashrender_set_env(hashrender_t* h, const float* env, uint32_t He, uint32_t We, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (!env || He == 0 || We == 0 || He > 8192 || We > 16384) return fail(h, HR_ERR_INVALID_ARG, "set_env: bad env / size");
  const size_t bytes = (size_t)He * We * 3 * sizeof(float);
  if (bytes > h->env_cap) {
    cudaFree(h->d_env); h->d_env = nullptr; h->env_cap = 0;
    cudaFree(h->d_env4); h->d_env4 = nullptr;
    HR_CUDA(h, cudaMalloc(&h->d_env, bytes));
    HR_CUDA(h, cudaMalloc(&h->d_env4, (size_t)He * We * sizeof(float4)));
    h->env_cap = bytes;
  }
  HR_CUDA(h, cudaMemcpyAsync(h->d_env, env, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  {
    const size_t n = (size_t)He * We;
    const size_t blocks = (n + 255) / 256;
    k_env_pack<<<(int)(blocks < 4096 ? blocks : 4096), 256, 0, (cudaStream_t)stream>>>(h->d_env, h->d_env4, n);
    h->launches++;
    HR_CUDA(h, cudaGetLastError());
  }
  h->env.env = h->d_env; h->env.env4 = h->d_env4; h->env.He = He; h->env.We = We;
  h->light_valid = false;
  return HR_OK;
}

int hashrender_encode(hashrender_t* h, const float* x, uint64_t N, float* feat, uint32_t* idx, float* w, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (N == 0) return HR_OK;
  if (!x || !feat) return fail(h, HR_ERR_INVALID_ARG, "encode: NULL x or feat");
  if (N > h->cfg.max_points) return fail(h, HR_ERR_INVALID_ARG, "encode: N exceeds max_points");
  const int grid = grid_for(h, N, 256, 8);
  if (h->grid.f16) k_encode<true><<<grid, 256, 0, (cudaStream_t)stream>>>(h->grid, x, N, feat, idx, w);
  else k_encode<false><<<grid, 256, 0, (cudaStream_t)stream>>>(h->grid, x, N, feat, idx, w);
  h->launches++;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

int hashrender_decode(hashrender_t* h, const float* feat, uint64_t N, float* brdf, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (N == 0) return HR_OK;
  if (!feat || !brdf) return fail(h, HR_ERR_INVALID_ARG, "decode: NULL feat or brdf");
  if (N > h->cfg.max_points) return fail(h, HR_ERR_INVALID_ARG, "decode: N exceeds max_points");
  k_decode_ffma<NT_FFMA><<<grid_for(h, N, NT_FFMA, 1), NT_FFMA, ffma_smem_bytes(NT_FFMA, false), (cudaStream_t)stream>>>(
      h->shade, h->d_wts, h->cfg.L * 2, feat, N, brdf);
  h->launches++;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

int hashrender_trace(hashrender_t* h, const float* x, const float* feat, uint64_t N, const hr_dirset* ds, float* vis, float* zv,
                     float* t, float* xsec, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (N == 0) return HR_OK;
  if (int e = check_dirset(h, ds, "trace", false)) return e;
  if (!vis || !t) return fail(h, HR_ERR_INVALID_ARG, "trace: NULL vis or t");
  if (!feat && !x) return fail(h, HR_ERR_INVALID_ARG, "trace: need x when feat is NULL (fused encode)");
  if (xsec && !x) return fail(h, HR_ERR_INVALID_ARG, "trace: xsec needs x");
  if (N > h->cfg.max_points) return fail(h, HR_ERR_INVALID_ARG, "trace: N exceeds max_points");
  const DirsetP d = to_dev(*ds);
  // the tensor-core kernel runs the arithmetic of render_frame's direct / secondary queries for this model (fp16 activations,
  // or hi/lo split precision for fp32 models), so v, z_v, t, x' of the production path are checked stage by stage
  if (const int path = render_path(h)) {
    h->last_path = path == 1 ? "tcgen05-f16" : "tcgen05-f16x3";
    if (path == 1)
      HR_CUDA(h, wg::launch_trace_p0(h->grid.f16, h->grid, h->shade, h->h_wts_tc.data(), h->d_wts_tc, x, feat, N, d, vis, zv, t, xsec,
                                     h->num_sms, (cudaStream_t)stream));
    else
      HR_CUDA(h, wg::launch_trace_p1(h->grid.f16, h->grid, h->shade, h->h_wts_tc.data(), h->d_wts_tc, x, feat, N, d, vis, zv, t, xsec,
                                     h->num_sms, (cudaStream_t)stream));
    h->launches++;
    return HR_OK;
  }
  h->last_path = "ffma32";
  const int grid = grid_for(h, N, NT_FFMA, 1);
  const size_t smem = ffma_smem_bytes(NT_FFMA, false);
  if (h->grid.f16) k_trace_ffma<true, NT_FFMA><<<grid, NT_FFMA, smem, (cudaStream_t)stream>>>(h->grid, h->shade, h->d_wts, x, feat, N, d, vis, zv, t, xsec);
  else k_trace_ffma<false, NT_FFMA><<<grid, NT_FFMA, smem, (cudaStream_t)stream>>>(h->grid, h->shade, h->d_wts, x, feat, N, d, vis, zv, t, xsec);
  h->launches++;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

int hashrender_shade(hashrender_t* h, const float* brdf, const float* wo, uint64_t N, const hr_dirset* ds, const float* vis,
                     const float* Lind, uint32_t terms, float* rgb, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (N == 0) return HR_OK;
  if (int e = check_dirset(h, ds, "shade", true)) return e;
  if (!brdf || !wo || !vis || !rgb) return fail(h, HR_ERR_INVALID_ARG, "shade: NULL brdf / wo / vis / rgb");
  if ((terms & HR_TERM_DIRECT) && !ds->Lin && !h->env.env) return fail(h, HR_ERR_INVALID_ARG, "shade: no env map set and no Lin");
  if ((terms & ~3u) || terms == 0) return fail(h, HR_ERR_INVALID_ARG, "shade: bad terms");
  if (N > h->cfg.max_points) return fail(h, HR_ERR_INVALID_ARG, "shade: N exceeds max_points");
  k_shade<<<grid_for(h, N, 256, 8), 256, 0, (cudaStream_t)stream>>>(h->env, h->shade, brdf, wo, N, to_dev(*ds), vis, Lind, terms, rgb);
  h->launches++;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

static int check_frame(hashrender* h, const hr_frame* f, const float* rgb) {
  if (!f) return fail(h, HR_ERR_INVALID_ARG, "render_frame: NULL frame");
  if (f->N == 0) return HR_OK;
  if (!f->x || !f->wo || !rgb) return fail(h, HR_ERR_INVALID_ARG, "render_frame: NULL x / wo / rgb");
  if (f->N > h->cfg.max_points) return fail(h, HR_ERR_INVALID_ARG, "render_frame: N exceeds max_points");
  if (!(f->flags & (HR_DIRECT | HR_INDIRECT)) || (f->flags & ~15u)) return fail(h, HR_ERR_INVALID_ARG, "render_frame: bad flags");
  bool need_env = false;
  if (f->flags & HR_DIRECT) {
    if (int e = check_dirset(h, &f->direct, "render_frame.direct", true)) return e;
    need_env |= !f->direct.Lin;
  }
  if (f->flags & HR_INDIRECT) {
    if (int e = check_dirset(h, &f->secondary, "render_frame.secondary", true)) return e;
    if (int e = check_dirset(h, &f->tertiary, "render_frame.tertiary", true)) return e;
    if (f->tertiary.S > kMaxS2) return fail(h, HR_ERR_UNSUPPORTED, "render_frame: tertiary S > 64");
    need_env |= !f->tertiary.Lin;
  }
  if (need_env && !h->env.env) return fail(h, HR_ERR_INVALID_ARG, "render_frame: no env map set and no Lin");
  return HR_OK;
}

int hashrender_render_frame(hashrender_t* h, const hr_frame* f, float* rgb, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (int e = check_frame(h, f, rgb)) return e;
  if (f->N == 0) return HR_OK;
  FrameP fr;
  fr.N = f->N; fr.x = f->x; fr.brdf = f->brdf; fr.wo = f->wo; fr.mask = f->mask; fr.flags = f->flags;
  fr.d = to_dev(f->direct); fr.s = to_dev(f->secondary); fr.t = to_dev(f->tertiary);
  if (!(f->flags & HR_DIRECT)) fr.d.S = 0;
  if (!(f->flags & HR_INDIRECT)) { fr.s.S = 0; fr.t.S = 0; }
  const int path = render_path(h);
  if (path && wg::frame_ok(fr)) {
    h->last_path = path == 1 ? "tcgen05-f16" : "tcgen05-f16x3";
    if (path == 1)
      HR_CUDA(h, wg::launch_p0(h->grid.f16, h->grid, h->env, h->shade, h->h_wts_tc.data(), h->d_wts_tc, h->d_wts, fr, rgb, h->d_ring, h->d_counters,
                               h->num_sms, (cudaStream_t)stream));
    else
      HR_CUDA(h, wg::launch_p1(h->grid.f16, h->grid, h->env, h->shade, h->h_wts_tc.data(), h->d_wts_tc, h->d_wts, fr, rgb, h->d_ring, h->d_counters,
                               h->num_sms, (cudaStream_t)stream));
    h->launches++;
    return HR_OK;
  }
  h->last_path = "ffma32";
  const int grid = grid_for(h, f->N, NT_FFMA, 1);
  const size_t smem = ffma_smem_bytes(NT_FFMA, true);
  if (h->grid.f16) k_render_ffma<true, NT_FFMA><<<grid, NT_FFMA, smem, (cudaStream_t)stream>>>(h->grid, h->env, h->shade, h->d_wts, fr, rgb);
  else k_render_ffma<false, NT_FFMA><<<grid, NT_FFMA, smem, (cudaStream_t)stream>>>(h->grid, h->env, h->shade, h->d_wts, fr, rgb);
  h->launches++;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

// Host-buffer variant.  The frame is cut into up to 8 row chunks: chunk c+1 is copied host->device on an internal copy stream
// while chunk c renders on the caller's stream, so the end-to-end time is max(copy, render) instead of their sum.
int hashrender_render_frame_host(hashrender_t* h, const hr_frame* f, float* rgb, void* stream, uint64_t* h2d_bytes, uint64_t* d2h_bytes) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (h2d_bytes) *h2d_bytes = 0;
  if (d2h_bytes) *d2h_bytes = 0;
  if (int e = check_frame(h, f, rgb)) return e;
  if (f->N == 0) return HR_OK;
  cudaStream_t st = (cudaStream_t)stream;
  if (!h->copy_stream) {
    HR_CUDA(h, cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 9; ++i) HR_CUDA(h, cudaEventCreateWithFlags(&h->ev[i], cudaEventDisableTiming));
  }
  const uint64_t N = f->N;
  const uint64_t wave = (uint64_t)h->num_sms * 4 * 128;              // pixels one pass of the render kernel's warpgroups covers
  int nchunks = (int)(N / (2 * wave));
  nchunks = nchunks < 1 ? 1 : (nchunks > 8 ? 8 : nchunks);
  const uint64_t rows_per = ((N + nchunks - 1) / nchunks + 127) / 128 * 128;

  // one entry per array that travels: `rows` rows of `row_elems` elements (the last row holds `last_elems`), elem bytes
  struct Arr { const char* src; char* dst; uint64_t rows, row_bytes, last_bytes, per_point; };
  Arr arr[16];
  int na = 0, slot = 0;
  uint64_t up = 0;
  auto ensure = [&](int s, size_t bytes) -> char* {
    if (bytes > h->stage_cap[s]) {
      cudaFree(h->stage[s]); h->stage[s] = nullptr; h->stage_cap[s] = 0;
      if (cudaMalloc(&h->stage[s], bytes) != cudaSuccess) return nullptr;
      h->stage_cap[s] = bytes;
    }
    return (char*)h->stage[s];
  };
  bool oom = false;
  // per_point = rows of this array per primary point (S_i for per-secondary-point tertiary sets, else 1; 0 = shared, copied once)
  auto add = [&](const void* src, uint64_t rows, uint64_t row_bytes, uint64_t last_bytes, uint64_t per_point) -> const void* {
    const int s = slot++;
    if (!src) return nullptr;
    const uint64_t total = (rows - 1) * row_bytes + last_bytes;
    char* d = ensure(s, total);
    if (!d) { oom = true; return nullptr; }
    arr[na++] = Arr{(const char*)src, d, rows, row_bytes, last_bytes, per_point};
    up += total;
    return d;
  };
  auto add_set = [&](const hr_dirset& d, uint64_t rows, uint64_t per_point, bool used) -> hr_dirset {
    hr_dirset o = d;
    if (!used) { slot += 3; return o; }
    if (d.point_stride) {
      o.dir = (const float*)add(d.dir, rows, d.point_stride * 4, 12ull * d.S, per_point);
      o.pdf = (const float*)add(d.pdf, rows, d.point_stride / 3 * 4, 4ull * d.S, per_point);
      o.Lin = (const float*)add(d.Lin, rows, d.point_stride * 4, 12ull * d.S, per_point);
    } else {
      o.dir = (const float*)add(d.dir, 1, 0, 12ull * d.S, 0);
      o.pdf = (const float*)add(d.pdf, 1, 0, 4ull * d.S, 0);
      o.Lin = (const float*)add(d.Lin, 1, 0, 12ull * d.S, 0);
    }
    return o;
  };
  hr_frame df = *f;
  df.x = (const float*)add(f->x, N, 12, 12, 1);
  df.brdf = (const float*)add(f->brdf, N, 28, 28, 1);
  df.wo = (const float*)add(f->wo, N, 12, 12, 1);
  df.mask = (const uint8_t*)add(f->mask, N, 1, 1, 1);
  df.direct = add_set(f->direct, N, 1, f->flags & HR_DIRECT);
  df.secondary = add_set(f->secondary, N, 1, f->flags & HR_INDIRECT);
  df.tertiary = add_set(f->tertiary, N * (uint64_t)f->secondary.S, f->secondary.S, f->flags & HR_INDIRECT);
  float* d_rgb = (float*)ensure(15, N * 12);
  if (oom || !d_rgb) return fail(h, HR_ERR_OOM, "render_frame_host: staging allocation failed");

  // the copy stream must not overwrite staging buffers an earlier call on `st` may still be reading
  HR_CUDA(h, cudaEventRecord(h->ev[8], st));
  HR_CUDA(h, cudaStreamWaitEvent(h->copy_stream, h->ev[8], 0));
  for (int c = 0; c < nchunks; ++c) {
    const uint64_t p0 = (uint64_t)c * rows_per, p1 = p0 + rows_per < N ? p0 + rows_per : N;
    if (p0 >= N) { nchunks = c; break; }
    for (int k = 0; k < na; ++k) {
      const Arr& a = arr[k];
      if (a.per_point == 0) {                                         // shared set: once, with the first chunk
        if (c == 0) HR_CUDA(h, cudaMemcpyAsync(a.dst, a.src, a.last_bytes, cudaMemcpyHostToDevice, h->copy_stream));
        continue;
      }
      const uint64_t r0 = p0 * a.per_point, r1 = p1 * a.per_point;
      const uint64_t bytes = r1 == a.rows ? (r1 - 1 - r0) * a.row_bytes + a.last_bytes : (r1 - r0) * a.row_bytes;
      HR_CUDA(h, cudaMemcpyAsync(a.dst + r0 * a.row_bytes, a.src + r0 * a.row_bytes, bytes, cudaMemcpyHostToDevice, h->copy_stream));
    }
    HR_CUDA(h, cudaEventRecord(h->ev[c], h->copy_stream));
  }
  for (int c = 0; c < nchunks; ++c) {
    const uint64_t p0 = (uint64_t)c * rows_per, p1 = p0 + rows_per < N ? p0 + rows_per : N;
    hr_frame cf = df;
    cf.N = p1 - p0;
    cf.x = df.x + 3 * p0;
    cf.wo = df.wo + 3 * p0;
    if (df.brdf) cf.brdf = df.brdf + 7 * p0;
    if (df.mask) cf.mask = df.mask + p0;
    auto off = [&](hr_dirset& d, uint64_t r0) {
      if (!d.point_stride) return;
      if (d.dir) d.dir += r0 * d.point_stride;
      if (d.pdf) d.pdf += r0 * (d.point_stride / 3);
      if (d.Lin) d.Lin += r0 * d.point_stride;
    };
    if (f->flags & HR_DIRECT) off(cf.direct, p0);
    if (f->flags & HR_INDIRECT) { off(cf.secondary, p0); off(cf.tertiary, p0 * (uint64_t)f->secondary.S); }
    HR_CUDA(h, cudaStreamWaitEvent(st, h->ev[c], 0));
    if (int e = hashrender_render_frame(h, &cf, d_rgb + 3 * p0, stream)) return e;
  }
  HR_CUDA(h, cudaMemcpyAsync(rgb, d_rgb, N * 12, cudaMemcpyDeviceToHost, st));
  HR_CUDA(h, cudaStreamSynchronize(st));
  if (h2d_bytes) *h2d_bytes = up;
  if (d2h_bytes) *d2h_bytes = N * 12;
  return HR_OK;
}

// Light-importance tables of the current env map (Q37): pmf over texels ~ luminance * sin(theta of the row centre), and
// its running sum rounded to fp32.  Built on the host in double (the map is a few KB), once per set_env.  Synchronises.
static int build_light_tables(hashrender* h, cudaStream_t st) {
  if (h->light_valid) return HR_OK;
  if (!h->env.env) return fail(h, HR_ERR_INVALID_ARG, "sample_mis: no env map set");
  const uint32_t He = h->env.He, We = h->env.We;
  const size_t n = (size_t)He * We;
  std::vector<float> env(n * 3), tab(2 * n);
  HR_CUDA(h, cudaStreamSynchronize(st));
  HR_CUDA(h, cudaMemcpy(env.data(), h->d_env, n * 12, cudaMemcpyDeviceToHost));
  std::vector<double> w(n);
  double tot = 0.0;
  for (uint32_t r = 0; r < He; ++r) {
    const double st_ = sin(3.14159265358979323846 * (r + 0.5) / He);
    for (uint32_t c = 0; c < We; ++c) {
      const float* p = &env[((size_t)r * We + c) * 3];
      const double Y = 0.2126 * (double)p[0] + 0.7152 * (double)p[1] + 0.0722 * (double)p[2];
      w[(size_t)r * We + c] = (Y > 0.0 ? Y : 0.0) * st_;
      tot += w[(size_t)r * We + c];
    }
  }
  if (!(tot > 0.0)) {
    tot = 0.0;
    for (uint32_t r = 0; r < He; ++r)
      for (uint32_t c = 0; c < We; ++c) { w[(size_t)r * We + c] = sin(3.14159265358979323846 * (r + 0.5) / He); tot += w[(size_t)r * We + c]; }
  }
  double run = 0.0;
  for (size_t k = 0; k < n; ++k) { const double q = w[k] / tot; run += q; tab[k] = (float)q; tab[n + k] = (float)run; }
  tab[2 * n - 1] = 1.0f;
  if (2 * n * 4 > h->light_cap) {
    cudaFree(h->d_light); h->d_light = nullptr; h->light_cap = 0;
    HR_CUDA(h, cudaMalloc(&h->d_light, 2 * n * 4));
    h->light_cap = 2 * n * 4;
  }
  HR_CUDA(h, cudaMemcpy(h->d_light, tab.data(), 2 * n * 4, cudaMemcpyHostToDevice));
  h->light_valid = true;
  return HR_OK;
}

int hashrender_sample_mis(hashrender_t* h, const float* brdf, const float* wo, uint64_t N, uint32_t spp, uint64_t seed, float* dir, float* pdf,
                          void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (N == 0) return HR_OK;
  if (!brdf || !wo || !dir || !pdf || spp == 0) return fail(h, HR_ERR_INVALID_ARG, "sample_mis: NULL brdf / wo / dir / pdf or spp == 0");
  if (N > h->cfg.max_points) return fail(h, HR_ERR_INVALID_ARG, "sample_mis: N exceeds max_points");
  if (int e = build_light_tables(h, (cudaStream_t)stream)) return e;
  smp::LightP lp;
  lp.pmf = h->d_light; lp.cdf = h->d_light + (size_t)h->env.He * h->env.We; lp.He = h->env.He; lp.We = h->env.We;
  const uint64_t total = N * spp;
  const uint64_t need = (total + 255) / 256, cap = (uint64_t)h->num_sms * 16;
  smp::k_sample_mis<<<(int)(need < cap ? need : cap), 256, 0, (cudaStream_t)stream>>>(lp, brdf, wo, N, spp, seed, dir, pdf);
  h->launches++;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

int hashrender_sample_stratified(hashrender_t* h, const float* normal, uint64_t rows, uint32_t Sa, uint32_t Sb, uint64_t seed, float* dir,
                                 float* pdf, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (rows == 0) return HR_OK;
  if (!dir || !pdf || Sa == 0 || Sb == 0) return fail(h, HR_ERR_INVALID_ARG, "sample_stratified: NULL dir / pdf or empty strata");
  const uint64_t total = rows * Sa * Sb;
  const uint64_t need = (total + 255) / 256, cap = (uint64_t)h->num_sms * 16;
  smp::k_sample_stratified<<<(int)(need < cap ? need : cap), 256, 0, (cudaStream_t)stream>>>(normal, rows, Sa, Sb, seed, dir, pdf);
  h->launches++;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

int hashrender_denoise(hashrender_t* h, const hr_denoise* d, float* out, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (!d) return fail(h, HR_ERR_INVALID_ARG, "denoise: NULL descriptor");
  if (d->H == 0 || d->W == 0) return HR_OK;
  if (!d->rgb || !d->normal || !d->pos || !out) return fail(h, HR_ERR_INVALID_ARG, "denoise: NULL rgb / normal / pos / out");
  if (d->iterations < 1 || d->iterations > 8) return fail(h, HR_ERR_INVALID_ARG, "denoise: iterations must be 1..8");
  if (!(d->sigma_z > 0.f) || !(d->sigma_l > 0.f) || !(d->sigma_n >= 0.f)) return fail(h, HR_ERR_INVALID_ARG, "denoise: bad sigma");
  const size_t n = (size_t)d->H * d->W;
  const size_t geo_b = n * sizeof(svgf::Geo), live_b = (n + 15) / 16 * 16, col_b = n * sizeof(float4);
  const size_t need = geo_b + live_b + 2 * col_b;
  if (need > h->svgf_cap) {
    cudaFree(h->d_svgf); h->d_svgf = nullptr; h->svgf_cap = 0;
    HR_CUDA(h, cudaMalloc(&h->d_svgf, need));
    h->svgf_cap = need;
  }
  char* base = (char*)h->d_svgf;
  svgf::Geo* geo = (svgf::Geo*)base;
  uint8_t* live = (uint8_t*)(base + geo_b);
  float4* colA = (float4*)(base + geo_b + live_b);
  float4* colB = colA + n;
  svgf::Params P;
  P.H = d->H; P.W = d->W; P.sigma_z = d->sigma_z; P.sigma_n = d->sigma_n; P.sigma_l = d->sigma_l;
  P.cam[0] = d->cam[0]; P.cam[1] = d->cam[1]; P.cam[2] = d->cam[2];
  cudaStream_t st = (cudaStream_t)stream;
  const uint64_t blocks = (n + 255) / 256, cap = (uint64_t)h->num_sms * 16;
  const int grid = (int)(blocks < cap ? blocks : cap);
  svgf::k_svgf_prep<<<grid, 256, 0, st>>>(P, d->rgb, d->albedo, d->pos, d->mask, geo, live, colA);
  svgf::k_svgf_variance<<<grid, 256, 0, st>>>(P, geo, d->normal, live, colA);
  float4* in = colA; float4* o = colB;
  for (uint32_t it = 0; it < d->iterations; ++it) {
    const bool last = it + 1 == d->iterations;
    svgf::k_svgf_atrous<<<grid, 256, 0, st>>>(P, 1 << it, geo, d->normal, live, in, last ? nullptr : o, d->albedo, last ? out : nullptr);
    float4* t = in; in = o; o = t;
  }
  h->launches += 2 + d->iterations;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

int hashrender_denoise_static(hashrender_t* h, const hr_denoise* d, float* out, void* stream) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (!d) return fail(h, HR_ERR_INVALID_ARG, "denoise_static: NULL descriptor");
  if (d->H == 0 || d->W == 0) return HR_OK;
  if (!d->rgb || !d->normal || !d->pos || !out) return fail(h, HR_ERR_INVALID_ARG, "denoise_static: NULL rgb / normal / pos / out");
  if (d->iterations < 1 || d->iterations > 8) return fail(h, HR_ERR_INVALID_ARG, "denoise_static: iterations must be 1..8");
  if (!(d->sigma_z > 0.f) || !(d->sigma_l > 0.f) || !(d->sigma_n >= 0.f)) return fail(h, HR_ERR_INVALID_ARG, "denoise_static: bad sigma");
  const size_t n = (size_t)d->H * d->W;
  if (n > kSvgfStaticPixels)
    return fail(h, HR_ERR_UNSUPPORTED, "denoise_static: %u x %u = %zu pixels exceed the static scratch (HASHRENDER_DENOISE_STATIC_MAX_PIXELS = %zu); "
                "use hashrender_denoise", d->H, d->W, n, kSvgfStaticPixels);
  char* base = nullptr;
  const cudaError_t eb = svgf_static_base(&base);
  if (eb != cudaSuccess || !base) return fail(h, HR_ERR_CUDA, "denoise_static: cudaGetSymbolAddress(g_svgf_static) failed: %s", cudaGetErrorString(eb));
  const size_t geo_b = n * sizeof(svgf::Geo), live_b = (n + 15) / 16 * 16;
  svgf::Geo* geo = (svgf::Geo*)base;
  uint8_t* live = (uint8_t*)(base + geo_b);
  float4* colA = (float4*)(base + geo_b + live_b);
  float4* colB = colA + n;
  svgf::Params P;
  P.H = d->H; P.W = d->W; P.sigma_z = d->sigma_z; P.sigma_n = d->sigma_n; P.sigma_l = d->sigma_l;
  P.cam[0] = d->cam[0]; P.cam[1] = d->cam[1]; P.cam[2] = d->cam[2];
  cudaStream_t st = (cudaStream_t)stream;
  const uint64_t blocks = (n + 255) / 256, cap = (uint64_t)h->num_sms * 16;
  const int grid = (int)(blocks < cap ? blocks : cap);
  svgf::k_svgf_prep<<<grid, 256, 0, st>>>(P, d->rgb, d->albedo, d->pos, d->mask, geo, live, colA);
  svgf::k_svgf_variance<<<grid, 256, 0, st>>>(P, geo, d->normal, live, colA);
  float4* in = colA; float4* o = colB;
  for (uint32_t it = 0; it < d->iterations; ++it) {
    const bool last = it + 1 == d->iterations;
    svgf::k_svgf_atrous<<<grid, 256, 0, st>>>(P, 1 << it, geo, d->normal, live, in, last ? nullptr : o, d->albedo, last ? out : nullptr);
    float4* t = in; in = o; o = t;
  }
  h->launches += 2 + d->iterations;
  HR_CUDA(h, cudaGetLastError());
  return HR_OK;
}

int hashrender_probe_gather(uint64_t table_bytes, uint32_t width, uint32_t group, uint32_t smem_bytes, double* loads_per_cycle_per_sm,
                            double* loads_per_s) {
  if (!loads_per_cycle_per_sm || !loads_per_s || table_bytes < 4096 || (table_bytes & (table_bytes - 1)) || table_bytes > (1ull << 33))
    return HR_ERR_INVALID_ARG;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return HR_ERR_CUDA;
  uint8_t* tab = nullptr; uint32_t* sink = nullptr; unsigned long long* cyc = nullptr;
  if (cudaMalloc(&tab, table_bytes) != cudaSuccess) return HR_ERR_OOM;
  cudaError_t e = cudaMalloc(&sink, 4);
  if (e == cudaSuccess) e = cudaMalloc(&cyc, 8);
  if (e == cudaSuccess) e = cudaMemset(tab, 1, table_bytes);
  int rc = HR_OK;
  if (e == cudaSuccess) {
    const int sm = (int)smem_bytes;
    if (width == 4 && group == 1) e = run_probe<4, 1>(tab, table_bytes, sm, sms, sink, cyc, loads_per_cycle_per_sm, loads_per_s);
    else if (width == 4 && group == 2) e = run_probe<4, 2>(tab, table_bytes, sm, sms, sink, cyc, loads_per_cycle_per_sm, loads_per_s);
    else if (width == 4 && group == 4) e = run_probe<4, 4>(tab, table_bytes, sm, sms, sink, cyc, loads_per_cycle_per_sm, loads_per_s);
    else if (width == 4 && group == 8) e = run_probe<4, 8>(tab, table_bytes, sm, sms, sink, cyc, loads_per_cycle_per_sm, loads_per_s);
    else if (width == 8 && group == 1) e = run_probe<8, 1>(tab, table_bytes, sm, sms, sink, cyc, loads_per_cycle_per_sm, loads_per_s);
    else if (width == 32 && group == 1) e = run_probe<32, 1>(tab, table_bytes, sm, sms, sink, cyc, loads_per_cycle_per_sm, loads_per_s);
    else rc = HR_ERR_UNSUPPORTED;
  }
  cudaFree(tab); cudaFree(sink); cudaFree(cyc);
  if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? HR_ERR_OOM : HR_ERR_CUDA;
  return rc;
}

int hashrender_table_layout(const hashrender_t* h, uint32_t* cell_major_levels, uint64_t* device_table_bytes) {
  if (!h) return HR_ERR_INVALID_ARG;
  if (cell_major_levels) *cell_major_levels = h->grid.nblock;
  if (device_table_bytes) *device_table_bytes = h->table_bytes;
  return HR_OK;
}

int hashrender_stats(hashrender_t* h, uint64_t* rays_traced, uint64_t* rays_evaluated, int reset) {
  if (!h) return HR_ERR_INVALID_ARG;
  unsigned long long c[4] = {0, 0, 0, 0};
  HR_CUDA(h, cudaDeviceSynchronize());
  HR_CUDA(h, cudaMemcpy(c, h->d_counters, sizeof(c), cudaMemcpyDeviceToHost));
  if (rays_traced) *rays_traced = c[2];
  if (rays_evaluated) *rays_evaluated = c[1];
  if (reset) HR_CUDA(h, cudaMemset(h->d_counters, 0, sizeof(c)));
  return HR_OK;
}

uint64_t hashrender_launch_count(const hashrender_t* h) { return h ? h->launches : 0; }
const char* hashrender_last_path(const hashrender_t* h) { return h ? h->last_path : "none"; }
const char* hashrender_last_error(const hashrender_t* h) { return h ? h->err : "NULL handle"; }

}  // extern "C"
