// fp32 build of the subdomain solve (subsystem (e)); see hz_sweep.cuh.
#include "hz_sweep_inst.cuh"

namespace hz {

// X(P, MX, MY, CSM, MAXT, MINB)
#define HZ_TILE_TABLE_F32(X) \
  X(1, 2, 2, 0, 1024, 1)     \
  X(1, 4, 4, 0, 512, 1)      \
  X(2, 1, 1, 0, 1024, 1)     \
  X(2, 2, 2, 0, 384, 1)      \
  X(3, 1, 1, 0, 512, 1)      \
  X(3, 2, 1, 0, 320, 1)      \
  X(3, 2, 1, 1, 576, 1)      \
  X(3, 2, 2, 1, 320, 1)      \
  X(4, 1, 1, 0, 384, 1)      \
  X(4, 1, 1, 1, 640, 1)

// W(P, M, CSM, MAXT, MINB): warp-specialised, square tiles
#define HZ_WS_TABLE_F32(W) \
  W(1, 2, 0, 1024, 1)      \
  W(1, 4, 0, 512, 1)       \
  W(2, 1, 0, 1024, 1)      \
  W(2, 2, 0, 384, 1)       \
  W(3, 1, 0, 128, 5)       \
  W(3, 1, 0, 256, 1)       \
  W(3, 1, 0, 512, 1)       \
  W(3, 2, 1, 320, 1)       \
  W(4, 1, 0, 384, 1)

// C(P, MX, MY, CL, MAXT, MINB): cluster of CL CTAs per subdomain, coefficients in registers
#define HZ_CL_TABLE_F32(C) \
  C(3, 1, 1, 2, 576, 1)    \
  C(3, 2, 1, 2, 320, 1)    \
  C(3, 2, 1, 4, 192, 1)    \
  C(3, 2, 1, 4, 192, 2)    \
  C(3, 1, 2, 2, 320, 1)    \
  C(3, 1, 1, 4, 320, 2)    \
  C(3, 1, 1, 8, 192, 3)    \
  C(3, 1, 1, 8, 640, 1)    \
  C(2, 2, 2, 2, 384, 1)    \
  C(2, 2, 2, 4, 384, 1)    \
  C(4, 1, 1, 2, 384, 1)    \
  C(4, 1, 1, 4, 384, 1)    \
  C(4, 1, 1, 16, 352, 1)

// K(P, M, MAXT): several small subdomains per block (hz_sweep_pack.cuh), square tiles
#define HZ_PK_TABLE_F32(K) \
  K(1, 4, 256)             \
  K(1, 2, 256)             \
  K(2, 2, 256)             \
  K(2, 1, 256)             \
  K(3, 1, 256)             \
  K(4, 1, 256)

// CW(P, MX, MY, CL, MAXT, MINB): cluster of CL CTAs per subdomain, warp-specialised edge pieces (hz_sweep_cw.cuh)
#define HZ_CW_TABLE_F32(CW) \
  CW(3, 2, 1, 2, 320, 1)   \
  CW(3, 2, 1, 4, 192, 1)   \
  CW(3, 2, 1, 8, 352, 1)   \
  CW(2, 2, 2, 4, 320, 1)   \
  CW(4, 1, 1, 4, 320, 1)   \
  CW(4, 1, 1, 16, 352, 1)

#define X_ENTRY(P, MX, MY, CSM, MAXT, MINB) \
  {P, MX, MY, CSM, MAXT, 0, MINB, 1, (const void *)k_sweep_tile<float, P, MX, MY, (CSM != 0), MAXT, MINB>},
#define W_ENTRY(P, M, CSM, MAXT, MINB) \
  {P, M, M, CSM, MAXT, 1, MINB, 1, (const void *)k_sweep_ws<float, P, M, (CSM != 0), MAXT, MINB>},
#define C_ENTRY(P, MX, MY, CL, MAXT, MINB) \
  {P, MX, MY, 0, MAXT, 0, MINB, CL, (const void *)k_sweep_cl<float, P, MX, MY, CL, MAXT, MINB>},
// K2(P, M, MAXT, MINB): two 64-tile subdomains per block sharing one edge warp (pk = 3).  Measured on config 5 against
// k_sweep_ws: p = 3 side 8 18.92 -> 17.39 ms, p = 1 side 32 11.33 -> 9.23 ms; p = 4 side 8 (19.50 -> 20.57) and p = 2
// side 16 (12.30 -> 12.67) are slower that way and keep k_sweep_ws.  Register cap of the p = 3 entry: 4 blocks per SM
// (96 registers) 17.39 ms, 3 blocks 18.31 ms, 5 blocks 20.90 ms
#define HZ_PK2_TABLE_F32(K2) \
  K2(3, 1, 160, 4)         \
  K2(1, 4, 160, 2)
#define K2_ENTRY(P, M, MAXT, MINB) \
  {P, M, M, 0, MAXT, 1, MINB, 1, (const void *)k_sweep_pack<float, P, M, MAXT, true, MINB, 9>, 3, 9},
// K4(P, M, MAXT, PRE): one subdomain of 16 x 16 tiles per block through the packed kernel (pk = 4: the corner node rides on
// the last top piece, so the 32 edge pieces fill ONE edge warp where k_sweep_ws needs two).  Measured on config 5 against
// k_sweep_ws: p = 1 side 64 12.83 -> 9.92 ms; p = 3 side 16 (18.74 -> 20.88), p = 4 side 16 (20.14 -> 21.11) and p = 2
// side 32 (12.23 -> 13.55) are slower and keep k_sweep_ws
#define HZ_PK4_TABLE_F32(K4, K4B) \
  K4B(3, 1, 288, true, 2)  \
  K4(1, 4, 288, false)
// K4B: the same with a register cap for MINB blocks per SM (and, in fp32, the FFMA2 updates)
#define K4B_ENTRY(P, M, MAXT, PRE, MINB) \
  {P, M, M, 0, MAXT, 1, MINB, 1, (const void *)k_sweep_pack<float, P, M, MAXT, PRE, MINB, 17>, 4, 17},
#define K4_ENTRY(P, M, MAXT, PRE) \
  {P, M, M, 0, MAXT, 1, 1, 1, (const void *)k_sweep_pack<float, P, M, MAXT, PRE, 1, 17>, 4, 17},
#define K_ENTRY(P, M, MAXT)                                                          \
  {P, M, M, 0, MAXT, 1, 1, 1, (const void *)k_sweep_pack<float, P, M, MAXT, false>, 1}, \
  {P, M, M, 0, MAXT, 1, 1, 1, (const void *)k_sweep_pack<float, P, M, MAXT, true>, 2},
#define CW_ENTRY(P, MX, MY, CL, MAXT, MINB) \
  {P, MX, MY, 0, MAXT, 1, MINB, CL, (const void *)k_sweep_cw<float, P, MX, MY, CL, MAXT, MINB>},
static const TileEntry kTilesF32[] = {HZ_CW_TABLE_F32(CW_ENTRY) HZ_WS_TABLE_F32(W_ENTRY) HZ_TILE_TABLE_F32(X_ENTRY) HZ_CL_TABLE_F32(C_ENTRY) HZ_PK_TABLE_F32(K_ENTRY) HZ_PK2_TABLE_F32(K2_ENTRY) HZ_PK4_TABLE_F32(K4_ENTRY, K4B_ENTRY)};
#undef K_ENTRY
#undef C_ENTRY
#undef X_ENTRY
#undef W_ENTRY
static const int kNumTilesF32 = sizeof(kTilesF32) / sizeof(kTilesF32[0]);

cudaError_t launch_sweep_dof_f32(const SweepArgs<float> &a, int p, SweepLaunch cfg, cudaStream_t st) {
  return launch_dof_impl<float>(a, p, cfg, st);
}
cudaError_t launch_sweep_tile_f32(const SweepArgs<float> &a, const TabC<float> *tc, int entry, SweepLaunch cfg,
                                  cudaStream_t st) {
  return launch_tile_impl<float>(kTilesF32, kNumTilesF32, a, tc, entry, cfg, st);
}
cudaError_t launch_sweep_stream_f32(const SweepArgs<float> &a, float *scr, int p, SweepLaunch cfg, cudaStream_t st) {
  return launch_stream_impl<float>(a, scr, p, cfg, st);
}
cudaError_t launch_minres_f32(const MinresArgs<float> &a, int p, SweepLaunch cfg, cudaStream_t st) {
  return launch_minres_impl<float>(a, p, cfg, st);
}
cudaError_t launch_minres_tile_f32(const MinresArgs<float> &a, const Elem1D<float> &ex1, const Elem1D<float> &ey1, int p, int m,
                                   SweepLaunch cfg, cudaStream_t st) {
  return launch_minres_tile_impl<float>(a, ex1, ey1, p, m, cfg, st);
}
int tile_table_f32(const TileEntry **out) {
  *out = kTilesF32;
  return kNumTilesF32;
}

}  // namespace hz
