// hz_sweep_inst.cuh — instantiation table and launch dispatch of the sweep kernels for one precision.
// Included by hz_sweep_f32.cu / hz_sweep_f64.cu (one translation unit per precision so they build in
// parallel).  HZ_TILE_TABLE(X) lists X(P, MX, MY, CSM, MAXT, MINB).
#pragma once
#include "hz_minres.cuh"
#include "hz_sweep.cuh"
#include "hz_sweep_stream.cuh"
#include "hz_sweep_cl.cuh"
#include "hz_sweep_cw.cuh"
#include "hz_sweep_pack.cuh"
#include "hz_sweep_tile.cuh"
#include "hz_sweep_ws.cuh"

namespace hz {

template <typename real>
static cudaError_t launch_dof_impl(const SweepArgs<real> &a, int p, SweepLaunch cfg, cudaStream_t st) {
  void (*fn)(const SweepArgs<real>) = nullptr;
  switch (p) {
    case 1: fn = k_sweep_dof<real, 1>; break;
    case 2: fn = k_sweep_dof<real, 2>; break;
    case 3: fn = k_sweep_dof<real, 3>; break;
    case 4: fn = k_sweep_dof<real, 4>; break;
    default: return cudaErrorInvalidValue;
  }
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
  if (e != cudaSuccess) return e;
  fn<<<cfg.blocks, cfg.threads, cfg.smem, st>>>(a);
  return cudaGetLastError();
}

template <typename real>
static cudaError_t launch_minres_impl(const MinresArgs<real> &a, int p, SweepLaunch cfg, cudaStream_t st) {
  void (*fn)(const MinresArgs<real>) = nullptr;
  switch (p) {
    case 1: fn = k_minres_dof<real, 1>; break;
    case 2: fn = k_minres_dof<real, 2>; break;
    case 3: fn = k_minres_dof<real, 3>; break;
    case 4: fn = k_minres_dof<real, 4>; break;
    default: return cudaErrorInvalidValue;
  }
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
  if (e != cudaSuccess) return e;
  fn<<<cfg.blocks, cfg.threads, cfg.smem, st>>>(a);
  return cudaGetLastError();
}

template <typename real>
static cudaError_t launch_minres_tile_impl(const MinresArgs<real> &a, const Elem1D<real> &ex1, const Elem1D<real> &ey1, int p, int m,
                                           SweepLaunch cfg, cudaStream_t st) {
  void (*fn)(const MinresArgs<real>, const Elem1D<real>, const Elem1D<real>) = nullptr;
  const int key = p * 10 + m;
  switch (key) {
    case 12: fn = k_minres_tile<real, 1, 2>; break;
    case 14: fn = k_minres_tile<real, 1, 4>; break;
    case 21: fn = k_minres_tile<real, 2, 1>; break;
    case 22: fn = k_minres_tile<real, 2, 2>; break;
    case 31: fn = k_minres_tile<real, 3, 1>; break;
    case 41: fn = k_minres_tile<real, 4, 1>; break;
    default: return cudaErrorInvalidValue;
  }
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
  if (e != cudaSuccess) return e;
  fn<<<cfg.blocks, cfg.threads, cfg.smem, st>>>(a, ex1, ey1);
  return cudaGetLastError();
}

template <typename real>
static cudaError_t launch_stream_impl(const SweepArgs<real> &a, real *scr, int p, SweepLaunch cfg, cudaStream_t st) {
  switch (p) {
    case 1: k_sweep_stream<real, 1><<<cfg.blocks, cfg.threads, 0, st>>>(a, scr); break;
    case 2: k_sweep_stream<real, 2><<<cfg.blocks, cfg.threads, 0, st>>>(a, scr); break;
    case 3: k_sweep_stream<real, 3><<<cfg.blocks, cfg.threads, 0, st>>>(a, scr); break;
    case 4: k_sweep_stream<real, 4><<<cfg.blocks, cfg.threads, 0, st>>>(a, scr); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

template <typename real>
static cudaError_t launch_tile_impl(const TileEntry *tab, int n, const SweepArgs<real> &a, const TabC<real> *tc, int entry,
                                    SweepLaunch cfg, cudaStream_t st) {
  if (entry < 0 || entry >= n || cfg.threads > tab[entry].maxt) return cudaErrorInvalidValue;
  const TileEntry &e = tab[entry];
  cudaError_t err = cudaFuncSetAttribute(e.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cfg.smem);
  if (err != cudaSuccess) return err;
  if (!tc) return cudaErrorInvalidValue;
  auto fn = reinterpret_cast<void (*)(const SweepArgs<real>, const TabC<real>)>(const_cast<void *>(e.fn));
  if (e.cl > 1) {  // one cluster of e.cl CTAs per subdomain
    if (e.cl > 8) {  // beyond the portable cluster size
      err = cudaFuncSetAttribute(e.fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
      if (err != cudaSuccess) return err;
    }
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3(cfg.blocks, 1, 1);
    lc.blockDim = dim3(cfg.threads, 1, 1);
    lc.dynamicSmemBytes = cfg.smem;
    lc.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = e.cl;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    lc.attrs = at;
    lc.numAttrs = 1;
    return cudaLaunchKernelEx(&lc, fn, a, *tc);
  }
  fn<<<cfg.blocks, cfg.threads, cfg.smem, st>>>(a, *tc);
  return cudaGetLastError();
}

}  // namespace hz
