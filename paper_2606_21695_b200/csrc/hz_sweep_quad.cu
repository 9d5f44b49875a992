// Instantiations and launch dispatch of the general-quadrilateral sweep kernel (hz_sweep_quad.cuh), both precisions.
#include "hz_sweep_quad.cuh"

namespace hz {

template <typename real>
static cudaError_t launch_quad_impl(const SweepArgs<real> &a, const QuadArgs<real> &q, const TabC<real> *tc, int p,
                                    SweepLaunch cfg, cudaStream_t st) {
  void (*fn)(const SweepArgs<real>, const QuadArgs<real>, const TabC<real>) = nullptr;
  const bool big = cfg.threads > 256;  // more than 256 elements per subdomain: 64-register cap
  switch (p) {
    case 1: fn = big ? k_sweep_quad<real, 1, 1024, 1> : k_sweep_quad<real, 1, 256, 1>; break;
    case 2: fn = big ? k_sweep_quad<real, 2, 1024, 1> : k_sweep_quad<real, 2, 256, 1>; break;
    case 3: fn = big ? k_sweep_quad<real, 3, 1024, 1> : k_sweep_quad<real, 3, 256, 1>; break;
    case 4: fn = big ? k_sweep_quad<real, 4, 1024, 1> : k_sweep_quad<real, 4, 256, 1>; break;
    default: return cudaErrorInvalidValue;
  }
  if (!tc || cfg.threads > 1024) return cudaErrorInvalidValue;
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
  if (e != cudaSuccess) return e;
  fn<<<cfg.blocks, cfg.threads, cfg.smem, st>>>(a, q, *tc);
  return cudaGetLastError();
}

cudaError_t launch_sweep_quad_f32(const SweepArgs<float> &a, const QuadArgs<float> &q, const TabC<float> *tc, int p,
                                  SweepLaunch cfg, cudaStream_t st) {
  return launch_quad_impl<float>(a, q, tc, p, cfg, st);
}
cudaError_t launch_sweep_quad_f64(const SweepArgs<double> &a, const QuadArgs<double> &q, const TabC<double> *tc, int p,
                                  SweepLaunch cfg, cudaStream_t st) {
  return launch_quad_impl<double>(a, q, tc, p, cfg, st);
}

}  // namespace hz
