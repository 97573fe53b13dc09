// hr_wg_p0.cu -- instantiations of k_render_wg for fp16 activations (mlp_dtype == HR_F16) + the weight-blob builder.
#include "hr_render_wg.cuh"
#include "hr_wg_api.h"

#ifndef HR_G_P0
#define HR_G_P0 4
#endif

namespace hr {
namespace wg {

void prepare_weights_blob(const hr_config& cfg, const float* brdf_w, const float* irt_w, std::vector<uint8_t>& out, size_t* const_bytes,
                          size_t* tile_bytes) {
  prepare_weights(cfg, brdf_w, irt_w, out);
  *const_bytes = sizeof(TcConst);
  *tile_bytes = out.size() - sizeof(TcConst);
}
size_t ring_bytes(int num_sms) { return (size_t)num_sms * kMaxG * kRing * sizeof(Item); }
bool frame_ok(const FrameP& fr) { return frame_supported(fr); }

cudaError_t launch_p0(bool f16tab, const GridP& g, const EnvP& env, const ShadeP& sp, const void* tc_const, const uint8_t* d_tiles,
                      const float* wts32, const FrameP& fr, float* rgb, void* ring, unsigned long long* counters, int num_sms, cudaStream_t st) {
  const TcConst& cw = *reinterpret_cast<const TcConst*>(tc_const);
  Item* rg = reinterpret_cast<Item*>(ring);
  const bool tsh = fr.t.stride == 0;
  if (f16tab) {
    if (tsh) return launch_one<true, 0, true, HR_G_P0>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
    return launch_one<true, 0, false, 2>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
  }
  if (tsh) return launch_one<false, 0, true, HR_G_P0>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
  return launch_one<false, 0, false, 2>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
}

cudaError_t launch_trace_p0(bool f16tab, const GridP& g, const ShadeP& sp, const void* tc_const, const uint8_t* d_tiles, const float* x,
                            const float* feat, unsigned long long N, const DirsetP& ds, float* vis, float* zv, float* t, float* xsec,
                            int num_sms, cudaStream_t st) {
  const TcConst& cw = *reinterpret_cast<const TcConst*>(tc_const);
  if (f16tab) return launch_trace_one<true, 0>(g, sp, cw, d_tiles, x, feat, N, ds, vis, zv, t, xsec, num_sms, st);
  return launch_trace_one<false, 0>(g, sp, cw, d_tiles, x, feat, N, ds, vis, zv, t, xsec, num_sms, st);
}

cudaError_t init_device_p0() {
  cudaError_t e;
  if ((e = render_attr<true, 0, true, HR_G_P0>()) != cudaSuccess) return e;
  if ((e = render_attr<true, 0, false, 2>()) != cudaSuccess) return e;
  if ((e = render_attr<false, 0, true, HR_G_P0>()) != cudaSuccess) return e;
  if ((e = render_attr<false, 0, false, 2>()) != cudaSuccess) return e;
  if ((e = trace_attr<true, 0>()) != cudaSuccess) return e;
  return trace_attr<false, 0>();
}

}  // namespace wg
}  // namespace hr
