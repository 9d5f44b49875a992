// fp64 build of the subdomain solve (subsystem (e)); see hz_sweep.cuh.
#include "hz_sweep_inst.cuh"

namespace hz {

// X(P, MX, MY, CSM, MAXT, MINB)
#define HZ_TILE_TABLE_F64(X) \
  X(1, 2, 2, 0, 1024, 1)     \
  X(1, 4, 4, 0, 256, 1)      \
  X(2, 1, 1, 0, 512, 1)      \
  X(2, 2, 2, 1, 320, 1)      \
  X(3, 1, 1, 0, 320, 1)      \
  X(3, 1, 1, 1, 512, 1)      \
  X(3, 2, 1, 1, 320, 1)      \
  X(4, 1, 1, 1, 320, 1)

// W(P, M, CSM, MAXT, MINB): warp-specialised, square tiles
#define HZ_WS_TABLE_F64(W) \
  W(1, 2, 0, 1024, 1)      \
  W(1, 4, 0, 256, 1)       \
  W(2, 1, 0, 512, 1)       \
  W(2, 2, 0, 128, 1)       \
  W(2, 2, 1, 320, 1)       \
  W(3, 1, 0, 128, 3)       \
  W(3, 1, 0, 128, 1)       \
  W(3, 1, 0, 320, 1)       \
  W(3, 1, 1, 512, 1)       \
  W(4, 1, 1, 128, 1)       \
  W(4, 1, 0, 128, 1)       \
  W(4, 1, 1, 320, 1)

// C(P, MX, MY, CL, MAXT, MINB): cluster of CL CTAs per subdomain, coefficients in registers
#define HZ_CL_TABLE_F64(C) \
  C(3, 1, 1, 2, 320, 1)    \
  C(3, 2, 1, 4, 192, 1)    \
  C(3, 2, 1, 8, 96, 2)    \
  C(3, 1, 1, 4, 320, 1)    \
  C(3, 1, 1, 8, 192, 2)    \
  C(3, 1, 1, 8, 320, 1)    \
  C(2, 1, 1, 2, 512, 1)    \
  C(2, 1, 1, 4, 512, 1)    \
  C(1, 2, 2, 2, 1024, 1)   \
  C(4, 1, 1, 4, 128, 1)    \
  C(4, 1, 1, 8, 128, 1)    \
  C(4, 1, 1, 8, 192, 1)    \
  C(2, 2, 2, 8, 192, 1)    \
  C(2, 1, 1, 8, 608, 1)    \
  C(3, 1, 1, 16, 352, 1)

// K(P, M, MAXT): several small subdomains per block (hz_sweep_pack.cuh), square tiles
#define HZ_PK_TABLE_F64(K) \
  K(1, 4, 256)             \
  K(1, 2, 256)             \
  K(2, 2, 256)             \
  K(2, 1, 256)             \
  K(3, 1, 256)             \
  K(4, 1, 256)

// CW(P, MX, MY, CL, MAXT, MINB): cluster of CL CTAs per subdomain, warp-specialised edge pieces (hz_sweep_cw.cuh)
#define HZ_CW_TABLE_F64(CW) \
  CW(3, 1, 1, 4, 320, 1)   \
  CW(1, 4, 4, 2, 192, 1)   \
  CW(3, 1, 1, 16, 352, 1)  \
  CW(2, 1, 1, 8, 608, 1)   \
  CW(4, 1, 1, 8, 192, 1)

#define X_ENTRY(P, MX, MY, CSM, MAXT, MINB) \
  {P, MX, MY, CSM, MAXT, 0, MINB, 1, (const void *)k_sweep_tile<double, P, MX, MY, (CSM != 0), MAXT, MINB>},
#define W_ENTRY(P, M, CSM, MAXT, MINB) \
  {P, M, M, CSM, MAXT, 1, MINB, 1, (const void *)k_sweep_ws<double, P, M, (CSM != 0), MAXT, MINB>},
#define C_ENTRY(P, MX, MY, CL, MAXT, MINB) \
  {P, MX, MY, 0, MAXT, 0, MINB, CL, (const void *)k_sweep_cl<double, P, MX, MY, CL, MAXT, MINB>},
// K2(P, M, MAXT, MINB): two 64-tile subdomains per block sharing one edge warp (pk = 3).  Measured on config 5 against
// k_sweep_ws: p = 3 side 8 37.27 -> 35.01 ms, p = 2 side 16 40.36 -> 37.30 ms; p = 4 side 8 (61.1 -> 64.7) and p = 1
// side 32 (26.0 -> 27.3) are slower that way and keep k_sweep_ws.  Register cap of the p = 3 entry: 2 blocks per SM
// (168 registers) 35.0 ms, 3 blocks 39.2 ms, uncapped 39.8 ms
#define HZ_PK2_TABLE_F64(K2) \
  K2(3, 1, 160, 2)         \
  K2(2, 2, 160, 1)
#define K2_ENTRY(P, M, MAXT, MINB) \
  {P, M, M, 0, MAXT, 1, MINB, 1, (const void *)k_sweep_pack<double, P, M, MAXT, true, MINB, 9>, 3, 9},
// K4(P, M, MAXT, PRE): one subdomain of 16 x 16 tiles per block through the packed kernel (pk = 4: the corner node rides on
// the last top piece, so the 32 edge pieces fill ONE edge warp where k_sweep_ws needs two).  Measured on config 5 against
// k_sweep_ws / k_sweep_cw: p = 3 side 16 38.15 -> 35.96 ms, p = 4 side 16 72.24 -> 68.09 ms (own part before the barrier),
// p = 1 side 64 34.84 (cluster of 2) -> 30.15 ms; p = 2 side 32 (35.51 -> 39.08) is slower and keeps k_sweep_ws
#define HZ_PK4_TABLE_F64(K4) \
  K4(3, 1, 288, false)     \
  K4(4, 1, 288, true)      \
  K4(1, 4, 288, true)
#define K4_ENTRY(P, M, MAXT, PRE) \
  {P, M, M, 0, MAXT, 1, 1, 1, (const void *)k_sweep_pack<double, P, M, MAXT, PRE, 1, 17>, 4, 17},
#define K_ENTRY(P, M, MAXT)                                                          \
  {P, M, M, 0, MAXT, 1, 1, 1, (const void *)k_sweep_pack<double, P, M, MAXT, false>, 1}, \
  {P, M, M, 0, MAXT, 1, 1, 1, (const void *)k_sweep_pack<double, P, M, MAXT, true>, 2},
#define CW_ENTRY(P, MX, MY, CL, MAXT, MINB) \
  {P, MX, MY, 0, MAXT, 1, MINB, CL, (const void *)k_sweep_cw<double, P, MX, MY, CL, MAXT, MINB>},
static const TileEntry kTilesF64[] = {HZ_CW_TABLE_F64(CW_ENTRY) HZ_WS_TABLE_F64(W_ENTRY) HZ_TILE_TABLE_F64(X_ENTRY) HZ_CL_TABLE_F64(C_ENTRY) HZ_PK_TABLE_F64(K_ENTRY) HZ_PK2_TABLE_F64(K2_ENTRY) HZ_PK4_TABLE_F64(K4_ENTRY)};
#undef K_ENTRY
#undef C_ENTRY
#undef X_ENTRY
#undef W_ENTRY
static const int kNumTilesF64 = sizeof(kTilesF64) / sizeof(kTilesF64[0]);

cudaError_t launch_sweep_dof_f64(const SweepArgs<double> &a, int p, SweepLaunch cfg, cudaStream_t st) {
  return launch_dof_impl<double>(a, p, cfg, st);
}
cudaError_t launch_sweep_tile_f64(const SweepArgs<double> &a, const TabC<double> *tc, int entry, SweepLaunch cfg,
                                  cudaStream_t st) {
  return launch_tile_impl<double>(kTilesF64, kNumTilesF64, a, tc, entry, cfg, st);
}
cudaError_t launch_sweep_stream_f64(const SweepArgs<double> &a, double *scr, int p, SweepLaunch cfg, cudaStream_t st) {
  return launch_stream_impl<double>(a, scr, p, cfg, st);
}
cudaError_t launch_minres_f64(const MinresArgs<double> &a, int p, SweepLaunch cfg, cudaStream_t st) {
  return launch_minres_impl<double>(a, p, cfg, st);
}
cudaError_t launch_minres_tile_f64(const MinresArgs<double> &a, const Elem1D<double> &ex1, const Elem1D<double> &ey1, int p, int m,
                                   SweepLaunch cfg, cudaStream_t st) {
  return launch_minres_tile_impl<double>(a, ex1, ey1, p, m, cfg, st);
}
int tile_table_f64(const TileEntry **out) {
  *out = kTilesF64;
  return kNumTilesF64;
}

}  // namespace hz
