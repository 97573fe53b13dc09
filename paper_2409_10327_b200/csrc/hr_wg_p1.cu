// hr_wg_p1.cu -- instantiations of k_render_wg in split precision (mlp_dtype == HR_F32 on the fp16 tensor cores).
#include "hr_render_wg.cuh"
#include "hr_wg_api.h"

#ifndef HR_G_P1
#define HR_G_P1 3
#endif

namespace hr {
namespace wg {

cudaError_t launch_p1(bool f16tab, const GridP& g, const EnvP& env, const ShadeP& sp, const void* tc_const, const uint8_t* d_tiles,
                      const float* wts32, const FrameP& fr, float* rgb, void* ring, unsigned long long* counters, int num_sms, cudaStream_t st) {
  const TcConst& cw = *reinterpret_cast<const TcConst*>(tc_const);
  Item* rg = reinterpret_cast<Item*>(ring);
  const bool tsh = fr.t.stride == 0;
  if (!((fr.flags & 4u) && fr.s.S && fr.t.S)) {                  // no indirect term: the direct-only kernel, four warpgroups per SM
    if (f16tab) return launch_one<true, 1, true, 4, false>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
    return launch_one<false, 1, true, 4, false>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
  }
  if (f16tab) {
    if (tsh) return launch_one<true, 1, true, HR_G_P1>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
    return launch_one<true, 1, false, 2>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
  }
  if (tsh) return launch_one<false, 1, true, HR_G_P1>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
  return launch_one<false, 1, false, 2>(g, env, sp, cw, d_tiles, wts32, fr, rgb, rg, counters, num_sms, st);
}

cudaError_t launch_trace_p1(bool f16tab, const GridP& g, const ShadeP& sp, const void* tc_const, const uint8_t* d_tiles, const float* x,
                            const float* feat, unsigned long long N, const DirsetP& ds, float* vis, float* zv, float* t, float* xsec,
                            int num_sms, cudaStream_t st) {
  const TcConst& cw = *reinterpret_cast<const TcConst*>(tc_const);
  if (f16tab) return launch_trace_one<true, 1>(g, sp, cw, d_tiles, x, feat, N, ds, vis, zv, t, xsec, num_sms, st);
  return launch_trace_one<false, 1>(g, sp, cw, d_tiles, x, feat, N, ds, vis, zv, t, xsec, num_sms, st);
}

cudaError_t init_device_p1() {
  cudaError_t e;
  if ((e = render_attr<true, 1, true, 4, false>()) != cudaSuccess) return e;
  if ((e = render_attr<false, 1, true, 4, false>()) != cudaSuccess) return e;
  if ((e = render_attr<true, 1, true, HR_G_P1>()) != cudaSuccess) return e;
  if ((e = render_attr<true, 1, false, 2>()) != cudaSuccess) return e;
  if ((e = render_attr<false, 1, true, HR_G_P1>()) != cudaSuccess) return e;
  if ((e = render_attr<false, 1, false, 2>()) != cudaSuccess) return e;
  if ((e = trace_attr<true, 1>()) != cudaSuccess) return e;
  return trace_attr<false, 1>();
}

}  // namespace wg
}  // namespace hr
