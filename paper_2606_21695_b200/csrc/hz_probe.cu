// hz_probe.cu -- bench-only micro-benchmark, built into its own library (libhz_probe.so), NOT part of the product
// ABI of include/hz.h: measures this GPU's CUDA-core FMA ceiling, which bench.py reports beside the derived
// roofline denominator.  No method arithmetic.
//
//   int hz_probe_fma(int kind, double *tflops, void *stream)
//     kind 0 = FP32 FMA, 1 = FP64 FMA; *tflops = best of 5 (2 flops per FMA); returns 0 on success.
#include <cuda_runtime.h>

namespace {

template <typename real>
__global__ void __launch_bounds__(256) k_probe_fma(int iters, real seed, real *out) {
  real a[16];
#pragma unroll
  for (int q = 0; q < 16; ++q) a[q] = seed + real(q) * real(1e-3) + real(threadIdx.x) * real(1e-6);
  const real m = real(0.999), c = real(1e-4);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
      for (int q = 0; q < 16; ++q) a[q] = a[q] * m + c;
  }
  real s = 0;
#pragma unroll
  for (int q = 0; q < 16; ++q) s += a[q];
  if (s == real(-12345)) out[0] = s;
}

}  // namespace

extern "C" int hz_probe_fma(int kind, double *result, void *stream) {
  if (!result || kind < 0 || kind > 1) return 1;
  cudaStream_t st = (cudaStream_t)stream;
  cudaDeviceProp prop;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return 3;
  const int sms = prop.multiProcessorCount;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return 3;
  float *d_out = nullptr;
  if (cudaMalloc((void **)&d_out, 64) != cudaSuccess) return 3;
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    float ms = 0.f;
    const int iters = kind == 0 ? 4096 : 2048, blocks = sms * 8, thr = 256;
    cudaEventRecord(e0, st);
    if (kind == 0) k_probe_fma<float><<<blocks, thr, 0, st>>>(iters, 1.0f, d_out);
    else k_probe_fma<double><<<blocks, thr, 0, st>>>(iters, 1.0, (double *)d_out);
    cudaEventRecord(e1, st);
    const double work = 2.0 * 64.0 * iters * (double)blocks * thr;
    if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) { cudaFree(d_out); return 3; }
    cudaEventElapsedTime(&ms, e0, e1);
    const double rate = work / (ms * 1e-3) / 1e12;
    if (rate > best) best = rate;
  }
  cudaFree(d_out);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *result = best;
  return 0;
}
