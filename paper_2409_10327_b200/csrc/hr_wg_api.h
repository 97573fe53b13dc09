// hr_wg_api.h -- host-callable entry points of the warpgroup-multiplexed tcgen05 render kernels (hr_render_wg.cuh).
// The kernels are instantiated in their own translation units (hr_wg_p0.cu: fp16 activations, hr_wg_p1.cu: split
// precision for fp32 models) so the library builds in parallel.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/hashrender.h"
#include "hr_device.cuh"

namespace hr {
namespace tc { struct TcConst; }
namespace wg {

// [ TcConst | hi tiles | lo tiles ]; const_bytes / tile_bytes give the split
void prepare_weights_blob(const hr_config& cfg, const float* brdf_w, const float* irt_w, std::vector<uint8_t>& out, size_t* const_bytes,
                          size_t* tile_bytes);
size_t ring_bytes(int num_sms);
bool frame_ok(const FrameP& fr);

// prec 0: fp16 activations; prec 1: hi/lo split activations and weights (fp32-grade).  counters: 4 x uint64 on the device.
cudaError_t launch_p0(bool f16tab, const GridP& g, const EnvP& env, const ShadeP& sp, const void* tc_const, const uint8_t* d_tiles,
                      const float* wts32, const FrameP& fr, float* rgb, void* ring, unsigned long long* counters, int num_sms, cudaStream_t st);
cudaError_t launch_p1(bool f16tab, const GridP& g, const EnvP& env, const ShadeP& sp, const void* tc_const, const uint8_t* d_tiles,
                      const float* wts32, const FrameP& fr, float* rgb, void* ring, unsigned long long* counters, int num_sms, cudaStream_t st);

// hashrender_trace (k_trace_wg): p0 = fp16 models, p1 = fp32 models in split precision (the arithmetic launch_p1 runs).
// feat == nullptr: the encode is fused; otherwise the caller's features [N, 2 L] are used and x is only needed for xsec.
cudaError_t launch_trace_p0(bool f16tab, const GridP& g, const ShadeP& sp, const void* tc_const, const uint8_t* d_tiles, const float* x,
                            const float* feat, unsigned long long N, const DirsetP& ds, float* vis, float* zv, float* t, float* xsec,
                            int num_sms, cudaStream_t st);
cudaError_t launch_trace_p1(bool f16tab, const GridP& g, const ShadeP& sp, const void* tc_const, const uint8_t* d_tiles, const float* x,
                            const float* feat, unsigned long long N, const DirsetP& ds, float* vis, float* zv, float* t, float* xsec,
                            int num_sms, cudaStream_t st);

// Opt-in of every kernel of the family to its dynamic shared-memory size, for the CURRENT device (hashrender_create calls both).
cudaError_t init_device_p0();
cudaError_t init_device_p1();

}  // namespace wg
}  // namespace hr
