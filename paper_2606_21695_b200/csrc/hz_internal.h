// hz_internal.h — types shared by the host driver (hz_api.cu) and the kernel translation units.
// Internal to the CUDA library; nothing here is visible through include/hz.h.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace hz {

constexpr int kMaxP = 4;
constexpr int kSideW = 0, kSideE = 1, kSideS = 2, kSideN = 3;

// Where node (i,j) of a subdomain lives inside the subdomain's slot range [0, NS).
//   variant 0 (one DOF per thread):   slot = j*lnx + i                       (thread = slot)
//   variant 2 (streamed fallback):    slot = j*lnx + i
//   variant 3 (general quads):        slot = j*lnx + i; ntx, nty = elements per subdomain side (one thread each)
//   variant 1 (register-blocked):     thread tile (tx,ty) owns TX x TY nodes; node (a,b) of the tile of
//                                     thread t = ty*ntx+tx lives at (b*TX+a)*NT + t, so that one node
//                                     index across the block's threads is one coalesced line.
struct Layout {
  int variant;
  int lnx, lny;  // nodes per subdomain side: ex*p+1, ey*p+1
  int TX, TY;    // nodes per thread tile (variant 1)
  int ntx, nty;  // thread tiles per side (variant 1): ex/MX+1, ey/MY+1
  int NT;        // threads per block
  int NS;        // slots per subdomain (>= lnx*lny; padding slots hold zeros)
  int cm;        // variant 1: 1 = virtual tiles numbered column by column, t = tx*nty+ty (cluster kernel: a column
                 // strip of the tile grid is then a contiguous range of t)
  __host__ __device__ inline int slot(int i, int j) const {
    if (variant != 1) return j * lnx + i;
    const int tx = i / TX, a = i - tx * TX, ty = j / TY, b = j - ty * TY;
    return (b * TX + a) * NT + (cm ? tx * nty + ty : ty * ntx + tx);
  }
};

// One row of the time-step tables (A0): cos(2 pi nu/N_t), sin(2 pi nu/N_t), kappa_nu, kappa_{nu+1/2}/omega.
template <typename real>
struct __align__(16) Tab4 {
  real c, s, k, kh;
};

// The whole time-step table as a by-value kernel parameter (constant bank): the step index is warp-uniform, so
// the kernel reads a row with uniform loads into uniform registers and the FMAs that use it keep a free
// vector-register read port.  Used by the warp-specialised kernel when n_t <= kTabCMax.
constexpr int kTabCMax = 256;
template <typename real>
struct TabC {
  Tab4<real> t[kTabCMax];
};

// 1-D element constants of the register-blocked kernel, already scaled by 4/h^2 and the GLL weights:
//   kin[a][c] = (4/h^2) K[a][c] / w_a        rows of element-interior nodes a = 1..P-1
//   k0[c]     = (4/h^2) K[0][c] / (2 w_0)    row of an element's first node (shared with the element before)
//   kp[c]     = (4/h^2) K[P][c] / (2 w_0)    row of an element's last node  (shared with the element after)
template <typename real>
struct Elem1D {
  real kin[kMaxP + 1][kMaxP + 1];
  real k0[kMaxP + 1];
  real kp[kMaxP + 1];
};

template <typename real>
struct SweepArgs {
  Layout lay;
  int sx, sy;      // subdomain grid
  int exq, exr, eyq, eyr;  // ragged partitions (general-quad kernel): see Geo
  int E;           // edge stride of lambda / g / kedge / bs arrays
  int n_t, n_wh, warm;
  real sigma, omega, cos_h, sin_h, two_over_nt;  // cos_h = cos(pi/N_t), sin_h = sin(pi/N_t)
  const Tab4<real> *tab;                         // [n_t]
  const real *gamma, *alpha, *bbf_re, *bbf_im;   // [L][NS]; bbf_im may be NULL
  real *u_sub;                                   // [L][2][NS]
  const real *lam;                               // [L][4][2][E]  lambda^n
  real *gout;                                    // [L][4][2][E]  outgoing g
  const real *k2edge;                            // [L][4][E]     2 k_j on each side
  const real *bs;                                // [L][4][E]     beta_j * s_j^{side}
  const real *bandx, *bandy;                     // variant 0: [lnx][2P+1], [lny][2P+1]
  Elem1D<real> ex1, ey1;                         // variant 1
  // fused exchange (optional): lam is then lambda^{n-1}, read-write; g_prev the neighbours' g^{n-1}
  int fused;
  int worder;  // warp-role order of the warp-specialised kernel (hz_sweep_ws.cuh): 0 bulk warps first, 1 / 2 see there
  real relax;
  const real *g_prev;
  real *lam_rw;
  int pack;  // packed small-subdomain kernel (hz_sweep_pack.cuh): subdomains per thread block
  int cmerge;  // packed kernel: 1 = the corner node rides on the last top piece's lane (one edge piece fewer per subdomain)
  int L;     // number of subdomains
};

// Extra arguments of the general-quadrilateral sweep kernel (hz_sweep_quad.cuh)
template <typename real>
struct QuadArgs {
  const real *G;                 // [L][3 (P+1)^2][nep]: w_a w_b {gxx, gxy, gyy} of every quadrature point
  int nep;                       // element stride of G (threads per block)
  real D[kMaxP + 1][kMaxP + 1];  // D[a][c] = l_c'(xi_a)
};

struct TileEntry {
  int p, mx, my, csm, maxt;  // csm: gamma / beta b in shared memory instead of registers
  int ws;                    // 1: warp-specialised kernel (hz_sweep_ws.cuh), needs mx == my
  int minb;                  // __launch_bounds__ min blocks per SM (register cap = 64K / (minb * maxt))
  int cl;                    // > 1: thread-block-cluster kernel (hz_sweep_cl.cuh), CTAs per subdomain
  const void *fn;
  int pk;                    // > 0: packed small-subdomain kernel (hz_sweep_pack.cuh), several subdomains per block;
                             // 2: its PRE instantiation (own part of a step before the block barrier)
                             // 3: two subdomains of up to 64 full tiles per block (one shared edge warp)
  int ntx;                   // pk = 3: > 0: compiled for ntx = nty = this many thread tiles per side
};

struct SweepLaunch {
  int blocks, threads;
  size_t smem;
};

// Implemented in hz_sweep_*.cu.  Return cudaErrorInvalidValue when no instantiation matches.
cudaError_t launch_sweep_dof_f32(const SweepArgs<float> &a, int p, SweepLaunch cfg, cudaStream_t st);
cudaError_t launch_sweep_dof_f64(const SweepArgs<double> &a, int p, SweepLaunch cfg, cudaStream_t st);
cudaError_t launch_sweep_tile_f32(const SweepArgs<float> &a, const TabC<float> *tc, int entry, SweepLaunch cfg,
                                  cudaStream_t st);
cudaError_t launch_sweep_tile_f64(const SweepArgs<double> &a, const TabC<double> *tc, int entry, SweepLaunch cfg,
                                  cudaStream_t st);
cudaError_t launch_sweep_stream_f32(const SweepArgs<float> &a, float *scr, int p, SweepLaunch cfg, cudaStream_t st);
cudaError_t launch_sweep_stream_f64(const SweepArgs<double> &a, double *scr, int p, SweepLaunch cfg, cudaStream_t st);
cudaError_t launch_sweep_quad_f32(const SweepArgs<float> &a, const QuadArgs<float> &q, const TabC<float> *tc, int p,
                                  SweepLaunch cfg, cudaStream_t st);
cudaError_t launch_sweep_quad_f64(const SweepArgs<double> &a, const QuadArgs<double> &q, const TabC<double> *tc, int p,
                                  SweepLaunch cfg, cudaStream_t st);
template <typename real>
struct MinresArgs;
cudaError_t launch_minres_f32(const MinresArgs<float> &a, int p, SweepLaunch cfg, cudaStream_t st);
cudaError_t launch_minres_f64(const MinresArgs<double> &a, int p, SweepLaunch cfg, cudaStream_t st);
// register-blocked MINRES (square tiles of m x m elements); cudaErrorInvalidValue when (p, m) is not compiled
cudaError_t launch_minres_tile_f32(const MinresArgs<float> &a, const Elem1D<float> &ex1, const Elem1D<float> &ey1, int p, int m,
                                   SweepLaunch cfg, cudaStream_t st);
cudaError_t launch_minres_tile_f64(const MinresArgs<double> &a, const Elem1D<double> &ex1, const Elem1D<double> &ey1, int p, int m,
                                   SweepLaunch cfg, cudaStream_t st);
// compiled register-blocked instantiations of one precision
int tile_table_f32(const TileEntry **out);
int tile_table_f64(const TileEntry **out);

}  // namespace hz
