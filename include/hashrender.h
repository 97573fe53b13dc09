/* hashrender.h -- C ABI of the B200-native recursively executed hash-grid renderer.
 *
 * The hot path of "Baking Relightable NeRF for Real-time Direct/Indirect Illumination Rendering"
 * (arXiv 2409.10327; citations are lines of /root/reference/PAPER.md): for every primary surface point x
 * and sampled light direction w_i, f = H(x) (multi-resolution hash-grid encoder), n,a,r = B(f)
 * (BRDF decoder MLP), v,t = I(f, w_i) (implicit ray tracer MLP: hard visibility + expected depth,
 * PAPER.md:80, 98), x' = x + t*w_i, the recursive re-evaluation at x' and
 * the Monte-Carlo rendering equation (Eq. 1) with the two-bounce incoming radiance
 * L = V*L_i + (1-V)*L'_o (Eq. 2).  Readings of points the paper leaves open are the Qn
 * entries of DESIGN.md.
 *
 * Conventions
 *  - Every function returns an int status (HR_OK = 0, ...); nothing throws or aborts across the ABI.
 *    hashrender_last_error(h) returns a NUL-terminated string owned by the handle (valid until the next
 *    failing call on that handle or its destruction).
 *  - Pointers are DEVICE pointers unless the comment says `host`.  All device work is enqueued
 *    asynchronously on the caller's cudaStream_t (passed as void*, NULL = legacy default stream).  Calls that
 *    synchronise: hashrender_create, hashrender_destroy, hashrender_render_frame_host (the stream, before it returns),
 *    hashrender_stats (the device) and the FIRST hashrender_sample_mis after a set_env (the stream, once: it reads the
 *    env map back to build the light tables on the host).  Nothing else synchronises.
 *  - Outputs are caller-allocated.  The library neither frees nor keeps caller memory after a call
 *    returns; hashrender_create COPIES (and re-lays-out / converts) tables and weights.
 *  - No allocation after create, except scratch that is created / grown on demand inside the handle and released by
 *    destroy: hashrender_render_frame_host's staging buffers, copy stream and events; hashrender_set_env's copy of the
 *    map (grown when a larger map arrives); hashrender_sample_mis's light tables; hashrender_denoise's image planes.
 *  - Alignment: every array 4-byte aligned; `feat` passed to hashrender_trace and `pdf` written by hashrender_sample_mis
 *    8-byte aligned (read / written as float2).
 *  - Arrays are row-major, innermost index last; float = IEEE binary32.  Directions and w_o are assumed
 *    unit length (not re-normalised).  Positions outside [0,1]^3 are clamped per component (Q6).
 *  - N == 0 is a no-op returning HR_OK.  NULL handle / NULL required pointer / S == 0 where a set is
 *    needed / unsupported shape => error status BEFORE any launch.
 *  - A handle is single-threaded; distinct handles are independent.
 *  - Supported shapes (else HR_ERR_UNSUPPORTED): F == 2, 1 <= L <= 16, 1 <= log2_T <= 28, hidden == 64,
 *    brdf_out == 7, irt_out == 2, tertiary S <= 64 (a shared tertiary set of more than 16 directions runs the fp32 FFMA kernels).
 */
#ifndef HASHRENDER_H_
#define HASHRENDER_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { HR_OK = 0, HR_ERR_INVALID_ARG = 1, HR_ERR_CUDA = 2, HR_ERR_OOM = 3, HR_ERR_UNSUPPORTED = 4 };
enum { HR_F32 = 0, HR_F16 = 1 };
enum { HR_DIRECT = 1, HR_SHADOW = 2, HR_INDIRECT = 4,             /* hr_frame.flags */
       HR_DENSE = 8 };  /* evaluate L'_o at EVERY secondary hit; default: only where its weight (1-v) f_r (n.w)^+ / p in
                           Eq. 2 is non-zero ("only occluded rays"); the result is the same */
enum { HR_TERM_DIRECT = 1, HR_TERM_INDIRECT = 2 };                /* hashrender_shade terms */
enum { HR_VIS_SOFT = 0, HR_VIS_HARD = 1 };
enum { HR_BRDF_LAMBERT = 0, HR_BRDF_DISNEY = 1 };

typedef struct hashrender hashrender_t;                           /* opaque */

/* Model description (14 levels, T = 2^17, F = 2, resolutions 16..131072, two 3-layer MLPs of
 * hidden width 64; BASELINE.json configs use L = 8/16, T = 2^14..2^24). */
typedef struct {
  uint32_t L, F, log2_T;
  const uint32_t* res;          /* host [L]: integer level resolutions N_l (Q2: given, never recomputed) */
  uint32_t table_dtype;         /* HR_F32 | HR_F16: storage type of the hash tables on the device */
  uint32_t mlp_dtype;           /* HR_F32: fp32 weights and activations (run on the fp16 tensor cores as hi + lo pairs, three
                                   passes, fp32-grade).  HR_F16: fp16 weights and hidden activations, fp32 accumulation of the
                                   64-wide layers; t, x' and the whole index path stay fp32; the final layer of visibility-only
                                   queries (direct shadow rays, tertiary rays) is summed with fp16x2 FMAs -- measured z_v error
                                   1.4e-4 (Q34) */
  uint32_t hidden;              /* 64 */
  uint32_t brdf_out, irt_out;   /* 7, 2 */
  float near_t, far_t;          /* 0.05, 1.5 */
  float rough_min;              /* 0.09 */
  float fresnel_f0;             /* 0.04 */
  uint32_t vis_mode;            /* HR_VIS_SOFT v = sigma(z_v) | HR_VIS_HARD v = [z_v > 0] (Q14) */
  uint32_t brdf_model;          /* HR_BRDF_LAMBERT | HR_BRDF_DISNEY (Q21) */
  float albedo_scale[3];        /* global albedo rescale; 1,1,1 = none */
  uint64_t max_points;          /* largest N any call will pass (sizes internal scratch) */
} hr_config;

/* A direction set (sampled w_i with its pdf).  dir[., S, 3], pdf[., S], optional Lin[., S, 3]
 * (incoming radiance per direction; NULL => looked up in the env map).  point_stride = number of floats of
 * `dir` (and of `Lin`) between consecutive points; pdf advances by point_stride / 3.  0 = ONE set shared by
 * all points (Q19). */
typedef struct {
  const float* dir; const float* pdf; const float* Lin;
  uint32_t S; uint64_t point_stride;
} hr_dirset;

/* One frame of primary points (the direct renderer G hands over material, normal and the
 * primary surface coordinate x). */
typedef struct {
  uint64_t N;
  const float* x;               /* [N,3] in [0,1]^3 */
  const float* brdf;            /* [N,7] = n(3) a(3) r(1), post-activation; NULL => B(H(x)) (Q30) */
  const float* wo;              /* [N,3] unit, towards the camera */
  const uint8_t* mask;          /* [N] nullable; 0 => rgb = 0 (Q27) */
  hr_dirset direct;             /* used with HR_DIRECT */
  hr_dirset secondary;          /* used with HR_INDIRECT: directions along which x' = x + t w is traced */
  hr_dirset tertiary;           /* used with HR_INDIRECT: directions sampled at every x' (8);
                                   point_stride != 0 => row index is i*secondary.S + j */
  uint32_t flags;               /* HR_DIRECT | HR_SHADOW | HR_INDIRECT [| HR_DENSE] */
} hr_frame;

/* Creates a renderer.  tables: host, fp32 [L][T][F] (every level owns T = 2^log2_T slots; a dense level --
 * (N_l+1)^3 <= T, Q3 -- uses the first (N_l+1)^3); converted once (RNE) when table_dtype == HR_F16.
 * brdf_w / irt_w: host, fp32 blobs, per layer W[out][in] row-major then b[out]; layers in->64->64->out with
 * in = L*F for B and L*F+3 ([f ; w], Q13) for I.  Synchronous.  Errors: INVALID_ARG, UNSUPPORTED, OOM, CUDA.
 * Device memory: the handle's copy of the tables is re-laid out for the gathers; the coarsest levels are also stored cell-major
 * (the 8 corner rows of every grid cell side by side: one or two 32-byte sectors per point and level instead of ~4.5), within a
 * budget of a quarter of the L2 cache when L*T rows fit the L2, else four times the size of the tables, and never more than a
 * quarter of the device memory free at the call (hashrender_table_layout reports what was built). */
int hashrender_create(const hr_config* cfg, const float* tables, const float* brdf_w, const float* irt_w,
                      hashrender_t** out);
int hashrender_destroy(hashrender_t* h);

/* Sets the equirect environment map, fp32 [He][We][3], DEVICE pointer; copied on `stream`. */
int hashrender_set_env(hashrender_t* h, const float* env, uint32_t He, uint32_t We, void* stream);

/* f = H(x) (steps a1-a4).  feat [N, L*F] fp32; optional idx [N, L, 8] uint32 (corner number
 * b0 + 2 b1 + 4 b2) and w [N, L, 3] fp32 (fractional position), both bit-exact against the oracle. */
int hashrender_encode(hashrender_t* h, const float* x, uint64_t N, float* feat, uint32_t* idx, float* w, void* stream);

/* n, a, r = B(f) (step a5).  feat [N, L*F] -> brdf [N, 7]. */
int hashrender_decode(hashrender_t* h, const float* feat, uint64_t N, float* brdf, void* stream);

/* v, t = I(f, w) for every direction of `ds` (step a6) and x' = clamp(x + t w) (
 * step a7).  feat NULL => the encode is fused (x required).  vis [N,S] (sigma(z_v) or {0,1}); zv nullable
 * [N,S] raw logit; t [N,S]; xsec nullable [N,S,3] (x required). ds->pdf and ds->Lin are not read.
 * Runs the arithmetic hashrender_render_frame uses for its direct / secondary queries on this model (see
 * hashrender_last_path), so the production path's z_v, t, x' can be checked stage by stage. */
int hashrender_trace(hashrender_t* h, const float* x, const float* feat, uint64_t N, const hr_dirset* ds,
                     float* vis, float* zv, float* t, float* xsec, void* stream);

/* Eq. 1 with Eq. 2 per direction on ONE set (steps a9-a11):
 * rgb = 1/S sum_s [ (terms & DIRECT) v L_i + (terms & INDIRECT) (1-v) Lind ] f_r (n.w)^+ / p.
 * brdf [N,7]; wo [N,3]; vis [N,S]; Lind nullable [N,S,3] (= L'_o); rgb [N,3]. */
int hashrender_shade(hashrender_t* h, const float* brdf, const float* wo, uint64_t N, const hr_dirset* ds,
                     const float* vis, const float* Lind, uint32_t terms, float* rgb, void* stream);

/* The fused, timed path (all steps a1-a11): rgb [N,3] = direct (shadowed) + one-bounce indirect radiance. */
int hashrender_render_frame(hashrender_t* h, const hr_frame* frame, float* rgb, void* stream);

/* Same as hashrender_render_frame but EVERY pointer in `frame` and `rgb` is a HOST pointer (pinned memory
 * recommended): copies inputs host->device, renders, copies rgb device->host, synchronises `stream`.  Large frames are
 * cut into row chunks whose copies (on an internal stream) overlap the previous chunk's render.
 * h2d_bytes / d2h_bytes (nullable) receive the bytes moved. */
int hashrender_render_frame_host(hashrender_t* h, const hr_frame* frame, float* rgb, void* stream,
                                 uint64_t* h2d_bytes, uint64_t* d2h_bytes);

/* On-device direction sampler (the step before the hot path; Q35-Q38).
 * sample_mis: per point i and sample s < spp, slot 2s = a light-importance ray (env-map luminance * sin(theta), stratified CDF
 * inversion, jittered in the texel), slot 2s+1 = a GGX visible-normal ray (alpha = roughness^2) about the normal of brdf[i]
 * ([N,7] = n a r, post-activation) for the view direction wo[i]; every ray carries the balance-heuristic pdf
 * (p_light + p_ggx) / 2, so the set plugs into hr_dirset with S = 2 spp.  dir [N, 2 spp, 3], pdf [N, 2 spp].  Needs set_env; the
 * first call after set_env builds the light tables on the host (synchronises `stream` once).  A pure function of
 * (env, brdf, wo, spp, seed): the generator is counter-based.
 * sample_stratified: Sa x Sb jittered strata per row, slot a*Sb + b; normal [rows,3] != NULL: cosine-weighted hemisphere about
 * normal[row] (pdf cos/pi); NULL: whole sphere (pdf 1/4pi).  dir [rows, Sa*Sb, 3], pdf [rows, Sa*Sb]. */
int hashrender_sample_mis(hashrender_t* h, const float* brdf, const float* wo, uint64_t N, uint32_t spp, uint64_t seed, float* dir,
                          float* pdf, void* stream);
int hashrender_sample_stratified(hashrender_t* h, const float* normal, uint64_t rows, uint32_t Sa, uint32_t Sb, uint64_t seed,
                                 float* dir, float* pdf, void* stream);

/* Spatial-only SVGF denoiser, the step after the path (SVGF on the raw MC result with the temporal parts removed;
 * depth gradient by finite differences of the depth derived from the primary surface coordinates; Q39-Q44).
 * Image arrays are row-major [H][W][.] DEVICE pointers.  rgb / out [H,W,3]; albedo [H,W,3] nullable (given => the illumination
 * rgb / max(albedo, 1e-3) is filtered and re-multiplied); normal [H,W,3] unit; pos [H,W,3] primary surface points, depth = |pos - cam|;
 * mask [H,W] nullable (0 => output 0, the pixel contributes to nobody).  iterations 1..8 a-trous passes (5: the published filter);
 * sigma_z 1, sigma_n 128, sigma_l 4 are the published edge-stopping parameters.  Scratch is grown on demand inside the handle. */
typedef struct {
  uint32_t H, W;
  const float* rgb; const float* albedo; const float* normal; const float* pos;
  float cam[3];
  const uint8_t* mask;
  uint32_t iterations;
  float sigma_z, sigma_n, sigma_l;
} hr_denoise;
int hashrender_denoise(hashrender_t* h, const hr_denoise* d, float* out, void* stream);

/* hashrender_denoise for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): the same kernels, arguments and result, with the image planes in a fixed array inside the library
 * (a file-scope __device__ array, 31.4 MB, held by every GPU that loads the library until the process exits) instead of
 * handle-owned scratch.  Calls no cudaMalloc / cudaFree or allocating library routine; enqueues 2 + iterations kernels on
 * `stream` and returns.  H * W > HASHRENDER_DENOISE_STATIC_MAX_PIXELS (one 800 x 800 frame) => HR_ERR_UNSUPPORTED before any
 * launch, the message naming the limit.  The array's device address is looked up once per device (hashrender_create on that
 * device does it; otherwise the first call).  The array is SHARED by every call and every handle on the device and keeps the
 * last call's contents (each call overwrites all it reads, nothing needs clearing): two calls that overlap on the GPU --
 * different streams without an ordering between them, or two handles from two threads -- race on it and corrupt both results;
 * order them on one stream or with events. */
#define HASHRENDER_DENOISE_STATIC_MAX_PIXELS 640000
int hashrender_denoise_static(hashrender_t* h, const hr_denoise* d, float* out, void* stream);

/* Secondary-ray accounting of the render_frame calls since the last reset: rays_traced = secondary
 * (point, direction) rays whose (v, t) were evaluated, rays_evaluated = those whose L'_o was evaluated (all of them with
 * HR_DENSE).  Both nullable.  Synchronises the device.  Only the tcgen05 paths count; the FFMA path leaves both at 0. */
int hashrender_stats(hashrender_t* h, uint64_t* rays_traced, uint64_t* rays_evaluated, int reset);

/* Layout of the handle's device copy of the tables: how many of the coarsest levels are stored cell-major (see hashrender_create)
 * and the bytes the copy takes.  Both nullable. */
int hashrender_table_layout(const hashrender_t* h, uint32_t* cell_major_levels, uint64_t* device_table_bytes);

/* Measurement aid, no handle: the rate at which the current device serves fully divergent global loads -- the roofline of the
 * hash-grid gathers.  512 threads per SM draw pseudo-random slots of a scratch table of `table_bytes`
 * (a power of two, 4 KiB .. 8 GiB; allocated and freed inside the call) and load `group` consecutive words of `width` bytes
 * from each: (width, group) = (4,1) (8,1) (32,1) one load per 32-byte sector, (4,2) (4,4) (4,8) that many loads per sector.
 * smem_bytes of dynamic shared memory are requested, which sets the L1 left beside it.  Outputs (host): loads per SM clock
 * cycle and SM, loads per second for the chip.  Synchronous.  Errors: INVALID_ARG, UNSUPPORTED (other width / group), OOM, CUDA. */
int hashrender_probe_gather(uint64_t table_bytes, uint32_t width, uint32_t group, uint32_t smem_bytes,
                            double* loads_per_cycle_per_sm, double* loads_per_s);

/* Number of kernels this handle has launched so far (for launch accounting in benchmarks). */
uint64_t hashrender_launch_count(const hashrender_t* h);

/* Which implementation the last render_frame / trace used: "ffma32" (fp32 FFMA), "tcgen05-f16" (fp16 activations) or
 * "tcgen05-f16x3" (fp32 model on the fp16 tensor cores: activations and weights split hi + lo, three MMA passes, fp32
 * accumulate; chosen when tables, weights and activation bounds fit the fp16 range, else "ffma32"). Never NULL. */
const char* hashrender_last_path(const hashrender_t* h);

const char* hashrender_last_error(const hashrender_t* h);

/* ---- The step before the path: the CNN direct-illumination renderer G (Fig. 2, 90-96, 134; Q45-Q51) --------
 * "The direct illumination renderer G takes rays as input and outputs the material, normal, and primary surface coordinates"
 * (PAPER.md:80): one forward pass turns the ray map gamma = [o, d_down] of an h x w pixel array into full-resolution
 * (8h x 8w) maps, written straight into the arrays hr_frame takes.  Architecture: 1x1 conv-norm-act stem (6 -> width), n_res 1x1
 * conv-norm-act layers in residual blocks of two (x <- x + L2(L1(x))), three super-resolution blocks (bilinear x2, two 3x3
 * conv-norm-act layers with sr_ch[s] channels, 1x1 output mapping to 11 channels) joined by the output skip; norm = instance
 * normalisation with affine parameters (eps 1e-5, biased variance), act = exact GELU; output channels [n3 a3 r1 x3 mask1] with the
 * maps n/||n||, sigma(a), rough_min + (1 - rough_min) sigma(r), x = sigma(.), mask = [. > 0].  The paper's model: width 256,
 * n_res 28, sr_ch 128/64/32, h = w = 100.
 * Every convolution is a tcgen05 implicit GEMM fed by TMA; activations travel as fp16 hi + lo pairs with fp32 accumulation and fp32
 * normalisation / GELU / residual / upsampling, so the result is fp32-grade.  Convolution weights must be fp16-representable.
 * weights: host, fp32, per layer W[Cout][Cin][k][k], b[Cout] and (conv-norm-act layers) gamma[Cout], beta[Cout], in the order stem,
 * residual layers, then per block conv a, conv b, output mapping.  create is synchronous and allocates every buffer (about
 * 1 GB at the paper's size); forward only enqueues kernels on `stream`.  Supported (else HR_ERR_UNSUPPORTED): width a multiple of
 * 64 up to 256, n_res even, sr_ch[s] = 32 or a multiple of 64 up to 256. */
typedef struct hr_gnet hr_gnet_t;
typedef struct {
  uint32_t h, w;                /* ray array ("downsampled pixel array"), h w <= 65536; the output image is 8h x 8w */
  uint32_t width, n_res;        /* 256, 28 */
  uint32_t sr_ch[3];            /* 128, 64, 32 */
  float rough_min;              /* 0.09 */
} hr_gnet_config;
int hashrender_gbuffer_create(const hr_gnet_config* cfg, const float* weights, uint64_t n_weights, hr_gnet_t** out);
int hashrender_gbuffer_destroy(hr_gnet_t* h);
/* rays: DEVICE [h][w][6].  Outputs (DEVICE, each nullable, N = 64 h w pixels in row-major image order): x [N,3], brdf [N,7] = n a r
 * (post-activation: hr_frame.x / hr_frame.brdf), mask [N] (hr_frame.mask), raw [N,11] (the network's outputs before the maps). */
int hashrender_gbuffer_forward(hr_gnet_t* h, const float* rays, float* x, float* brdf, uint8_t* mask, float* raw, void* stream);
/* kernels launched so far; algorithmic flops of one forward (2 N Cout Cin k^2 per convolution, one pass, padding not counted) */
uint64_t hashrender_gbuffer_launch_count(const hr_gnet_t* h);
double hashrender_gbuffer_flops(const hr_gnet_t* h);
const char* hashrender_gbuffer_last_error(const hr_gnet_t* h);

#ifdef __cplusplus
}
#endif
#endif /* HASHRENDER_H_ */
