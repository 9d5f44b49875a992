// hz3_api.cu — C-ABI entry points of include/hz3.h: the 3-D hexahedral variant.
// Host-side setup (GLL tables, time-step tables, partition) and the outer driver on one stream.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/hz3.h"
#include "hz3_kernels.cuh"
#include "hz_host_gll.h"

using namespace hz;

struct hz3_ctx {
  Geo3 g{};
  Gll gll;
  double c_max = 0;
  int prec = 0, L = 0, n_t = 0;
  bool part = false;
  double dt = 0;
  double *d_c = nullptr, *d_fre = nullptr, *d_fim = nullptr, *d_bc = nullptr;
  void *d_tab = nullptr, *d_gamma = nullptr, *d_alpha = nullptr, *d_bre = nullptr, *d_bim = nullptr;
  void *d_usub = nullptr, *d_lam = nullptr, *d_g = nullptr, *d_k2 = nullptr, *d_bs = nullptr;
  void *d_bx = nullptr, *d_by = nullptr, *d_bz = nullptr;
  double *d_wx = nullptr, *d_wy = nullptr, *d_wz = nullptr, *d_part = nullptr, *d_red = nullptr, *d_u64 = nullptr;
  int threads = 0, colz = 0;  // colz > 0: column kernel with colz nodes per thread
  size_t smem = 0, ws_bytes = 0;
  BandZ<float> bz32{};
  BandZ<double> bz64{};
  TabC<float> tc32{};
  TabC<double> tc64{};
  std::string err;
};

namespace {

std::string g3_setup_error;

hz_status fail3(hz3_ctx *ctx, hz_status st, const std::string &msg) {
  if (ctx) ctx->err = msg; else g3_setup_error = msg;
  return st;
}
hz_status cuda_fail3(hz3_ctx *ctx, cudaError_t e, const char *what) {
  return fail3(ctx, e == cudaErrorMemoryAllocation ? HZ_ENOMEM : HZ_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define HZ3_CUDA(call)                                         \
  do {                                                         \
    cudaError_t e_ = (call);                                   \
    if (e_ != cudaSuccess) return cuda_fail3(ctx, e_, #call);  \
  } while (0)

inline int roundup3(int a, int b) { return (a + b - 1) / b * b; }

void free_partition3(hz3_ctx *c) {
  void **ptrs[] = {&c->d_tab, &c->d_gamma, &c->d_alpha, &c->d_bre, &c->d_bim, &c->d_usub, &c->d_lam, &c->d_g, &c->d_k2,
                   &c->d_bs, &c->d_bx, &c->d_by, &c->d_bz, (void **)&c->d_wx, (void **)&c->d_wy, (void **)&c->d_wz,
                   (void **)&c->d_part, (void **)&c->d_red, (void **)&c->d_u64};
  for (void **q : ptrs) { if (*q) cudaFree(*q); *q = nullptr; }
  c->part = false;
}

template <typename real>
cudaError_t upload3(const std::vector<double> &src, void **dst) {
  std::vector<real> tmp(src.begin(), src.end());
  cudaError_t e = cudaMalloc(dst, tmp.size() * sizeof(real));
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, tmp.data(), tmp.size() * sizeof(real), cudaMemcpyHostToDevice);
}

template <typename real>
Sweep3Args<real> make_args3(const hz3_ctx *c, const hz3_solve_opts *o) {
  Sweep3Args<real> a{};
  a.g = c->g;
  a.n_t = c->n_t; a.n_wh = o->n_wh; a.warm = o->warm_start;
  a.sigma = (real)c->g.sigma; a.omega = (real)c->g.omega;
  a.cos_h = (real)std::cos(M_PI / c->n_t); a.sin_h = (real)std::sin(M_PI / c->n_t);
  a.two_over_nt = (real)(2.0 / c->n_t);
  a.tab = (const Tab4<real> *)c->d_tab;
  a.gamma = (const real *)c->d_gamma; a.alpha = (const real *)c->d_alpha;
  a.bbf_re = (const real *)c->d_bre; a.bbf_im = (const real *)c->d_bim;
  a.u_sub = (real *)c->d_usub; a.lam = (const real *)c->d_lam; a.gout = (real *)c->d_g;
  a.k2face = (const real *)c->d_k2; a.bs = (const real *)c->d_bs;
  a.bandx = (const real *)c->d_bx; a.bandy = (const real *)c->d_by; a.bandz = (const real *)c->d_bz;
  return a;
}

template <typename real>
cudaError_t launch_sweep3(const hz3_ctx *c, const hz3_solve_opts *o, const TabC<real> &tc, cudaStream_t st) {
  void (*fn)(const Sweep3Args<real>, const TabC<real>) = nullptr;
  // register cap by block size (the node's 3(2P+1) band coefficients live in registers)
  const int sel = c->threads <= 256 ? 0 : (c->threads <= 512 ? 1 : 2);
#define HZ3_CASE(P_)                                                                                            \
  case P_:                                                                                                      \
    fn = sel == 0 ? k3_sweep_dof<real, P_, 256> : (sel == 1 ? k3_sweep_dof<real, P_, 512> : k3_sweep_dof<real, P_, 1024>); \
    break;
  switch (c->g.p) {
    HZ3_CASE(1)
    HZ3_CASE(2)
    HZ3_CASE(3)
    HZ3_CASE(4)
    default: return cudaErrorInvalidValue;
  }
#undef HZ3_CASE
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem);
  if (e != cudaSuccess) return e;
  fn<<<c->L, c->threads, c->smem, st>>>(make_args3<real>(c, o), tc);
  return cudaGetLastError();
}

// compiled (P, LNZ) pairs of the column kernel: LNZ = ez*P + 1 for the block shapes of PAPER.md:265
bool col_supported(int P, int lnz) {
  switch (P) {
    case 1: return lnz == 3 || lnz == 5 || lnz == 9;
    case 2: return lnz == 5 || lnz == 9;
    case 3: return lnz == 4 || lnz == 7 || lnz == 10;
    case 4: return lnz == 5 || lnz == 9;
    default: return false;
  }
}

template <typename real>
cudaError_t launch_sweep3_col(const hz3_ctx *c, const hz3_solve_opts *o, const BandZ<real> &bz, const TabC<real> &tc,
                              cudaStream_t st) {
  void (*fn)(const Sweep3Args<real>, const BandZ<real>, const TabC<real>) = nullptr;
  const int key = c->g.p * 100 + c->colz;
#define HZ3_COL(P_, Z_) \
  case P_ * 100 + Z_: fn = k3_sweep_col<real, P_, Z_, 128>; break;
  switch (key) {
    HZ3_COL(1, 3) HZ3_COL(1, 5) HZ3_COL(1, 9)
    HZ3_COL(2, 5) HZ3_COL(2, 9)
    HZ3_COL(3, 4) HZ3_COL(3, 7) HZ3_COL(3, 10)
    HZ3_COL(4, 5) HZ3_COL(4, 9)
    default: return cudaErrorInvalidValue;
  }
#undef HZ3_COL
  cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem);
  if (e != cudaSuccess) return e;
  fn<<<c->L, c->threads, c->smem, st>>>(make_args3<real>(c, o), bz, tc);
  return cudaGetLastError();
}

hz_status residual3_impl(hz3_ctx *ctx, const void *u_dev, int prec, double *rel, cudaStream_t st) {
  const Geo3 &g = ctx->g;
  const long long total = (long long)g.npx * g.npy * g.npz;
  const int nb = (int)((total + 255) / 256);
  if (!ctx->d_part) {
    HZ3_CUDA(cudaMalloc((void **)&ctx->d_part, (size_t)2 * nb * sizeof(double)));
    HZ3_CUDA(cudaMalloc((void **)&ctx->d_red, 2 * sizeof(double)));
  }
  const double *u64 = (const double *)u_dev;
  if (prec == HZ_F32) {
    if (!ctx->d_u64) HZ3_CUDA(cudaMalloc((void **)&ctx->d_u64, (size_t)2 * total * sizeof(double)));
    k3_to_f64<float><<<(unsigned)((2 * total + 255) / 256), 256, 0, st>>>((const float *)u_dev, ctx->d_u64, 2 * total);
    HZ3_CUDA(cudaGetLastError());
    u64 = ctx->d_u64;
  }
  Ref1D ref{};
  for (int a = 0; a <= g.p; ++a) {
    ref.w[a] = ctx->gll.w[a];
    for (int b = 0; b <= g.p; ++b) ref.K[a][b] = ctx->gll.K[a][b];
  }
  k3_residual<double><<<nb, 256, 0, st>>>(g, ref, ctx->d_c, ctx->d_fre, ctx->d_fim, ctx->d_bc, u64, const_cast<double *>(u64),
                                          ctx->d_part);
  HZ3_CUDA(cudaGetLastError());
  k_reduce2<<<1, 1024, 0, st>>>(ctx->d_part, nb, ctx->d_red);
  HZ3_CUDA(cudaGetLastError());
  double h[2];
  HZ3_CUDA(cudaMemcpyAsync(h, ctx->d_red, sizeof(h), cudaMemcpyDeviceToHost, st));
  HZ3_CUDA(cudaStreamSynchronize(st));
  *rel = h[1] > 0.0 ? std::sqrt(h[0] / h[1]) : std::sqrt(h[0]);
  return HZ_OK;
}

}  // namespace

extern "C" {

hz_status hz3_mesh_setup(hz3_ctx **out, int nx, int ny, int nz, const double *box, int p, const double *c_nodes,
                         double omega, const double *f_re, const double *f_im, const double *bc_lambda) {
  hz3_ctx *ctx = nullptr;
  if (!out || !box || !c_nodes || !f_re) return fail3(nullptr, HZ_EINVAL, "hz3_mesh_setup: NULL out, box, c_nodes or f_re");
  if (nx < 1 || ny < 1 || nz < 1 || !(box[3] > box[0]) || !(box[4] > box[1]) || !(box[5] > box[2]) || !(omega > 0.0) ||
      !std::isfinite(omega))
    return fail3(nullptr, HZ_EINVAL, "hz3_mesh_setup: need nx,ny,nz >= 1, a non-degenerate box, omega > 0");
  if (p < 1 || p > kMaxP) return fail3(nullptr, HZ_EUNSUPPORTED, "hz3_mesh_setup: degree p must be 1..4");
  const long long nn = ((long long)nx * p + 1) * ((long long)ny * p + 1) * ((long long)nz * p + 1);
  if (nn > (1ll << 31) - 1) return fail3(nullptr, HZ_EUNSUPPORTED, "hz3_mesh_setup: more than 2^31-1 nodes");
  double cmax = 0.0;
  for (long long q = 0; q < nn; ++q) {
    if (!(c_nodes[q] > 0.0) || !std::isfinite(c_nodes[q])) return fail3(nullptr, HZ_EINVAL, "hz3_mesh_setup: c_nodes must be finite and > 0");
    cmax = std::fmax(cmax, c_nodes[q]);
  }
  hz3_ctx *c = new (std::nothrow) hz3_ctx();
  if (!c) return fail3(nullptr, HZ_ENOMEM, "hz3_mesh_setup: out of host memory");
  Geo3 &g = c->g;
  g.nx = nx; g.ny = ny; g.nz = nz; g.p = p; g.npx = nx * p + 1; g.npy = ny * p + 1; g.npz = nz * p + 1;
  g.hx = (box[3] - box[0]) / nx; g.hy = (box[4] - box[1]) / ny; g.hz = (box[5] - box[2]) / nz; g.omega = omega;
  g.FB = std::max(g.npy * g.npz, std::max(g.npx * g.npz, g.npx * g.npy));
  c->c_max = cmax;
  make_gll(p, &c->gll);
  const size_t bytes = (size_t)nn * sizeof(double);
  cudaError_t e = cudaMalloc((void **)&c->d_c, bytes);
  if (e == cudaSuccess) e = cudaMalloc((void **)&c->d_fre, bytes);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_c, c_nodes, bytes, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_fre, f_re, bytes, cudaMemcpyHostToDevice);
  if (e == cudaSuccess && f_im) {
    e = cudaMalloc((void **)&c->d_fim, bytes);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_fim, f_im, bytes, cudaMemcpyHostToDevice);
  }
  if (e == cudaSuccess && bc_lambda) {
    e = cudaMalloc((void **)&c->d_bc, (size_t)12 * g.FB * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpy(c->d_bc, bc_lambda, (size_t)12 * g.FB * sizeof(double), cudaMemcpyHostToDevice);
  }
  if (e != cudaSuccess) {
    hz_status st = cuda_fail3(nullptr, e, "hz3_mesh_setup (device allocation / copy)");
    hz3_destroy(c);
    return st;
  }
  (void)ctx;
  *out = c;
  return HZ_OK;
}

hz_status hz3_partition(hz3_ctx *ctx, int sx, int sy, int sz, hz_prec prec, double cfl_frac, int nodes_per_thread,
                        hz3_part_info *info) {
  if (!ctx) return HZ_EINVAL;
  Geo3 &g = ctx->g;
  if (sx < 1 || sy < 1 || sz < 1 || g.nx % sx || g.ny % sy || g.nz % sz)
    return fail3(ctx, HZ_EINVAL, "hz3_partition: sx, sy, sz must be >= 1 and divide nx, ny, nz");
  if (prec != HZ_F32 && prec != HZ_F64) return fail3(ctx, HZ_EINVAL, "hz3_partition: bad precision");
  if (!(cfl_frac > 0.0) || cfl_frac > 1.0) return fail3(ctx, HZ_EINVAL, "hz3_partition: cfl_frac must be in (0,1]");
  free_partition3(ctx);
  const int P = g.p;
  g.sx = sx; g.sy = sy; g.sz = sz; g.ex = g.nx / sx; g.ey = g.ny / sy; g.ez = g.nz / sz;
  g.lnx = g.ex * P + 1; g.lny = g.ey * P + 1; g.lnz = g.ez * P + 1;
  const int N = g.lnx * g.lny * g.lnz;
  if (N > 1024) return fail3(ctx, HZ_EUNSUPPORTED, "hz3_partition: one node per thread needs <= 1024 nodes per subdomain");
  g.NS = roundup3(N, 32);
  g.F = std::max(g.lny * g.lnz, std::max(g.lnx * g.lnz, g.lnx * g.lny));
  ctx->L = sx * sy * sz; ctx->prec = prec;
  const size_t rs = prec == HZ_F32 ? 4 : 8;
  // time step (reading R9 in 3-D)
  const double lmax = ctx->c_max * ctx->c_max * ctx->gll.lambda_p * (1.0 / (g.hx * g.hx) + 1.0 / (g.hy * g.hy) + 1.0 / (g.hz * g.hz));
  const double T = 2.0 * M_PI / g.omega;
  int n_t = (int)std::ceil(T / (cfl_frac * 2.0 / std::sqrt(lmax)) * (1.0 - 1e-12));
  if (n_t < 4) n_t = 4;
  ctx->n_t = n_t; ctx->dt = T / n_t;
  g.theta = std::tan(g.omega * ctx->dt / 2.0) / g.omega;
  g.sigma = std::sin(g.omega * ctx->dt / 2.0) / (g.omega / 2.0);
  ctx->threads = g.NS;
  ctx->colz = 0;
  if (nodes_per_thread != 1 && col_supported(P, g.lnz) && g.lnx * g.lny <= 128) {
    ctx->colz = g.lnz;
    ctx->threads = roundup3(g.lnx * g.lny, 32);
  }
  ctx->smem = 2 * (size_t)((N + 2 * P * (g.lnx * g.lny + g.lnx + 1) + 3) / 4 * 4) * rs;  // see k3_sweep_dof
  if (ctx->smem > 227 * 1024) return fail3(ctx, HZ_EUNSUPPORTED, "hz3_partition: subdomain volume exceeds shared memory");
  std::vector<double> tab((size_t)n_t * 4);
  const double tan2 = std::tan(M_PI / n_t) * std::tan(M_PI / n_t);
  for (int nu = 0; nu < n_t; ++nu) {
    tab[4 * nu + 0] = std::cos(2.0 * M_PI * nu / n_t);
    tab[4 * nu + 1] = std::sin(2.0 * M_PI * nu / n_t);
    tab[4 * nu + 2] = std::cos(2.0 * M_PI * nu / n_t) - 0.25 + 0.25 * tan2;
    tab[4 * nu + 3] = (std::cos(2.0 * M_PI * (nu + 0.5) / n_t) - 0.25 + 0.25 * tan2) / g.omega;
  }
  for (int nu = 0; nu < n_t && nu < kTabCMax; ++nu) {
    ctx->tc32.t[nu] = Tab4<float>{(float)tab[4 * nu], (float)tab[4 * nu + 1], (float)tab[4 * nu + 2], (float)tab[4 * nu + 3]};
    ctx->tc64.t[nu] = Tab4<double>{tab[4 * nu], tab[4 * nu + 1], tab[4 * nu + 2], tab[4 * nu + 3]};
  }
  std::vector<double> bx, by, bz, wx, wy, wz;
  make_band(ctx->gll, g.ex, g.hx, &bx, &wx);
  make_band(ctx->gll, g.ey, g.hy, &by, &wy);
  make_band(ctx->gll, g.ez, g.hz, &bz, &wz);
  if (ctx->colz)
    for (int k = 0; k < g.lnz; ++k)
      for (int d = 0; d < 2 * P + 1; ++d) {
        ctx->bz32.z[k][d] = (float)bz[(size_t)k * (2 * P + 1) + d];
        ctx->bz64.z[k][d] = bz[(size_t)k * (2 * P + 1) + d];
      }
  const size_t LS = (size_t)ctx->L * g.NS, lam_n = (size_t)ctx->L * 12 * g.F, face_n = (size_t)ctx->L * 6 * g.F;
  size_t ws = 0;
  auto alloc0 = [&](void **ptr, size_t bytes) -> cudaError_t {
    cudaError_t e = cudaMalloc(ptr, bytes);
    if (e != cudaSuccess) return e;
    ws += bytes;
    return cudaMemset(*ptr, 0, bytes);
  };
  HZ3_CUDA(alloc0(&ctx->d_gamma, LS * rs));
  HZ3_CUDA(alloc0(&ctx->d_alpha, LS * rs));
  HZ3_CUDA(alloc0(&ctx->d_bre, LS * rs));
  if (ctx->d_fim || ctx->d_bc) HZ3_CUDA(alloc0(&ctx->d_bim, LS * rs));
  HZ3_CUDA(alloc0(&ctx->d_usub, 2 * LS * rs));
  HZ3_CUDA(alloc0(&ctx->d_lam, lam_n * rs));
  HZ3_CUDA(alloc0(&ctx->d_g, lam_n * rs));
  HZ3_CUDA(alloc0(&ctx->d_k2, face_n * rs));
  HZ3_CUDA(alloc0(&ctx->d_bs, face_n * rs));
  if (prec == HZ_F32) {
    HZ3_CUDA(upload3<float>(tab, &ctx->d_tab)); HZ3_CUDA(upload3<float>(bx, &ctx->d_bx));
    HZ3_CUDA(upload3<float>(by, &ctx->d_by)); HZ3_CUDA(upload3<float>(bz, &ctx->d_bz));
  } else {
    HZ3_CUDA(upload3<double>(tab, &ctx->d_tab)); HZ3_CUDA(upload3<double>(bx, &ctx->d_bx));
    HZ3_CUDA(upload3<double>(by, &ctx->d_by)); HZ3_CUDA(upload3<double>(bz, &ctx->d_bz));
  }
  HZ3_CUDA(upload3<double>(wx, (void **)&ctx->d_wx));
  HZ3_CUDA(upload3<double>(wy, (void **)&ctx->d_wy));
  HZ3_CUDA(upload3<double>(wz, (void **)&ctx->d_wz));
  const long long total = (long long)ctx->L * N;
  const unsigned nb = (unsigned)((total + 255) / 256);
  if (prec == HZ_F32)
    k3_build<float><<<nb, 256>>>(g, ctx->d_c, ctx->d_fre, ctx->d_fim, ctx->d_bc, ctx->d_wx, ctx->d_wy, ctx->d_wz,
                                 (float *)ctx->d_gamma, (float *)ctx->d_alpha, (float *)ctx->d_bre, (float *)ctx->d_bim,
                                 (float *)ctx->d_k2, (float *)ctx->d_bs);
  else
    k3_build<double><<<nb, 256>>>(g, ctx->d_c, ctx->d_fre, ctx->d_fim, ctx->d_bc, ctx->d_wx, ctx->d_wy, ctx->d_wz,
                                  (double *)ctx->d_gamma, (double *)ctx->d_alpha, (double *)ctx->d_bre,
                                  (double *)ctx->d_bim, (double *)ctx->d_k2, (double *)ctx->d_bs);
  HZ3_CUDA(cudaGetLastError());
  HZ3_CUDA(cudaDeviceSynchronize());
  ctx->ws_bytes = ws;
  ctx->part = true;
  if (info) {
    hz3_part_info inf{};
    inf.n_t = n_t; inf.dofs_per_sub = N; inf.lnx = g.lnx; inf.lny = g.lny; inf.lnz = g.lnz; inf.face_stride = g.F;
    inf.threads_per_block = ctx->threads; inf.blocks = ctx->L; inf.nodes_per_thread = ctx->colz ? ctx->colz : 1;
    inf.dt = ctx->dt; inf.theta = g.theta; inf.sigma = g.sigma;
    inf.smem_bytes = ctx->smem; inf.workspace_bytes = ws;
    *info = inf;
  }
  return HZ_OK;
}

hz_status hz3_ddm_solve(hz3_ctx *ctx, const hz3_solve_opts *opts, void *u_out, hz3_solve_info *info, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!opts) return fail3(ctx, HZ_EINVAL, "hz3_ddm_solve: NULL opts");
  if (!ctx->part) return fail3(ctx, HZ_ESTATE, "hz3_ddm_solve: call hz3_partition first");
  if (opts->n_outer < 0 || opts->n_wh < 1 || !(opts->relax > 0.0) || opts->relax > 1.0)
    return fail3(ctx, HZ_EINVAL, "hz3_ddm_solve: need n_outer >= 0, n_wh >= 1, relax in (0,1]");
  cudaStream_t st = (cudaStream_t)stream;
  const Geo3 &g = ctx->g;
  const size_t rs = ctx->prec == HZ_F32 ? 4 : 8;
  const size_t lam_n = (size_t)ctx->L * 12 * g.F;
  if (opts->reset_state) {
    HZ3_CUDA(cudaMemsetAsync(ctx->d_lam, 0, lam_n * rs, st));
    HZ3_CUDA(cudaMemsetAsync(ctx->d_g, 0, lam_n * rs, st));
    HZ3_CUDA(cudaMemsetAsync(ctx->d_usub, 0, (size_t)2 * ctx->L * g.NS * rs, st));
  }
  const int n = opts->n_outer;
  const bool checking = opts->tol > 0.0 && opts->check_every > 0;
  const long long total = (long long)g.npx * g.npy * g.npz;
  const unsigned nbg = (unsigned)((total + 255) / 256);
  if (checking && !ctx->d_u64) HZ3_CUDA(cudaMalloc((void **)&ctx->d_u64, (size_t)2 * total * sizeof(double)));
  std::vector<cudaEvent_t> ev((size_t)2 * n + 2);
  for (auto &e : ev) HZ3_CUDA(cudaEventCreate(&e));
  auto cleanup = [&]() { for (auto &e : ev) cudaEventDestroy(e); };
  cudaError_t ce = cudaSuccess;
  const unsigned nbx = (unsigned)((lam_n + 255) / 256);
  int done = 0, launches = 0;
  double rel = -1.0;
  ce = cudaEventRecord(ev[2 * n + 1], st);  // start of the call
  for (int it = 0; it < n && ce == cudaSuccess; ++it) {
    ce = cudaEventRecord(ev[2 * it], st);
    if (ce == cudaSuccess) {
      if (ctx->colz)
        ce = ctx->prec == HZ_F32 ? launch_sweep3_col<float>(ctx, opts, ctx->bz32, ctx->tc32, st)
                                 : launch_sweep3_col<double>(ctx, opts, ctx->bz64, ctx->tc64, st);
      else
        ce = ctx->prec == HZ_F32 ? launch_sweep3<float>(ctx, opts, ctx->tc32, st) : launch_sweep3<double>(ctx, opts, ctx->tc64, st);
    }
    if (ce == cudaSuccess) ce = cudaEventRecord(ev[2 * it + 1], st);
    if (ce != cudaSuccess) break;
    if (ctx->prec == HZ_F32) k3_exchange<float><<<nbx, 256, 0, st>>>(g, (float)opts->relax, (float *)ctx->d_lam, (const float *)ctx->d_g);
    else k3_exchange<double><<<nbx, 256, 0, st>>>(g, opts->relax, (double *)ctx->d_lam, (const double *)ctx->d_g);
    ce = cudaGetLastError();
    if (ce != cudaSuccess) break;
    ++done; launches += 2;
    if (checking && (done % opts->check_every == 0 || done == n)) {  // the only reduction, outside the sweep
      if (ctx->prec == HZ_F32) k3_gather<float, double><<<nbg, 256, 0, st>>>(g, (const float *)ctx->d_usub, ctx->d_u64);
      else k3_gather<double, double><<<nbg, 256, 0, st>>>(g, (const double *)ctx->d_usub, ctx->d_u64);
      ce = cudaGetLastError();
      if (ce != cudaSuccess) break;
      hz_status rs_ = residual3_impl(ctx, ctx->d_u64, HZ_F64, &rel, st);
      launches += 3;
      if (rs_ != HZ_OK) { cleanup(); return rs_; }
      if (rel <= opts->tol) break;
    }
  }
  if (ce == cudaSuccess) ce = cudaEventRecord(ev[2 * n], st);
  if (ce == cudaSuccess && u_out) {
    if (ctx->prec == HZ_F32) k3_gather<float, float><<<nbg, 256, 0, st>>>(g, (const float *)ctx->d_usub, (float *)u_out);
    else k3_gather<double, double><<<nbg, 256, 0, st>>>(g, (const double *)ctx->d_usub, (double *)u_out);
    ce = cudaGetLastError();
    ++launches;
  }
  cudaEvent_t ev_end = nullptr;
  if (ce == cudaSuccess) ce = cudaEventCreate(&ev_end);
  if (ce == cudaSuccess) ce = cudaEventRecord(ev_end, st);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
  if (ce != cudaSuccess) { cleanup(); if (ev_end) cudaEventDestroy(ev_end); return cuda_fail3(ctx, ce, "hz3_ddm_solve"); }
  double sw = 0.0, ex = 0.0;
  for (int it = 0; it < done; ++it) {
    float a = 0.f, b = 0.f;
    cudaEventElapsedTime(&a, ev[2 * it], ev[2 * it + 1]);
    sw += a;
    if (!checking) {  // with residual checks in between, the exchange has no closing event of its own
      cudaEventElapsedTime(&b, ev[2 * it + 1], it + 1 < done ? ev[2 * it + 2] : ev[2 * n]);
      ex += b;
    }
  }
  float tot = 0.f;
  cudaEventElapsedTime(&tot, ev[2 * n + 1], ev_end);
  cudaEventDestroy(ev_end);
  cleanup();
  if (info) {
    info->n_outer_done = done; info->n_t = ctx->n_t; info->rel_residual = rel; info->total_ms = tot;
    info->sweep_ms_total = sw; info->exch_ms_total = checking ? -1.0 : ex;
    info->dof_timesteps = (double)done * ctx->L * (double)(g.lnx * g.lny * g.lnz) * opts->n_wh * (ctx->n_t - 1);
    info->launches = launches;
  }
  return HZ_OK;
}

hz_status hz3_residual(hz3_ctx *ctx, const void *u_dev, hz_prec prec, double *rel, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!u_dev || !rel) return fail3(ctx, HZ_EINVAL, "hz3_residual: NULL u_dev or rel");
  return residual3_impl(ctx, u_dev, prec, rel, (cudaStream_t)stream);
}

hz_status hz3_operator_time(hz3_ctx *ctx, const double *u_dev, int reps, double *ms_per_eval, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!u_dev || !ms_per_eval || reps < 1) return fail3(ctx, HZ_EINVAL, "hz3_operator_time: NULL argument or reps < 1");
  cudaStream_t st = (cudaStream_t)stream;
  const Geo3 &g = ctx->g;
  const long long total = (long long)g.npx * g.npy * g.npz;
  const int nb = (int)((total + 255) / 256);
  if (!ctx->d_part) {
    HZ3_CUDA(cudaMalloc((void **)&ctx->d_part, (size_t)2 * nb * sizeof(double)));
    HZ3_CUDA(cudaMalloc((void **)&ctx->d_red, 2 * sizeof(double)));
  }
  Ref1D ref{};
  for (int a = 0; a <= g.p; ++a) {
    ref.w[a] = ctx->gll.w[a];
    for (int b = 0; b <= g.p; ++b) ref.K[a][b] = ctx->gll.K[a][b];
  }
  cudaEvent_t e0, e1;
  HZ3_CUDA(cudaEventCreate(&e0));
  HZ3_CUDA(cudaEventCreate(&e1));
  k3_residual<double><<<nb, 256, 0, st>>>(g, ref, ctx->d_c, ctx->d_fre, ctx->d_fim, ctx->d_bc, u_dev, const_cast<double *>(u_dev), ctx->d_part);
  cudaEventRecord(e0, st);
  for (int r = 0; r < reps; ++r)
    k3_residual<double><<<nb, 256, 0, st>>>(g, ref, ctx->d_c, ctx->d_fre, ctx->d_fim, ctx->d_bc, u_dev, const_cast<double *>(u_dev), ctx->d_part);
  cudaEventRecord(e1, st);
  cudaError_t ce = cudaStreamSynchronize(st);
  float ms = 0.f;
  if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (ce != cudaSuccess) return cuda_fail3(ctx, ce, "hz3_operator_time");
  *ms_per_eval = ms / reps;
  return HZ_OK;
}

hz_status hz3_get_subdomain_state(hz3_ctx *ctx, double *u_sub, double *lam) {
  if (!ctx) return HZ_EINVAL;
  if (!ctx->part) return fail3(ctx, HZ_ESTATE, "hz3_get_subdomain_state: call hz3_partition first");
  const Geo3 &g = ctx->g;
  const long long n = std::max((long long)ctx->L * 2 * g.lnx * g.lny * g.lnz, (long long)ctx->L * 12 * g.F);
  const unsigned nb = (unsigned)((n + 255) / 256);
  if (ctx->prec == HZ_F32) k3_state_get<float><<<nb, 256>>>(g, (const float *)ctx->d_usub, (const float *)ctx->d_lam, u_sub, lam);
  else k3_state_get<double><<<nb, 256>>>(g, (const double *)ctx->d_usub, (const double *)ctx->d_lam, u_sub, lam);
  HZ3_CUDA(cudaGetLastError());
  HZ3_CUDA(cudaDeviceSynchronize());
  return HZ_OK;
}

const char *hz3_last_error(hz3_ctx *ctx) { return ctx ? ctx->err.c_str() : g3_setup_error.c_str(); }

void hz3_destroy(hz3_ctx *ctx) {
  if (!ctx) return;
  free_partition3(ctx);
  double **ptrs[] = {&ctx->d_c, &ctx->d_fre, &ctx->d_fim, &ctx->d_bc};
  for (double **q : ptrs) { if (*q) cudaFree(*q); *q = nullptr; }
  delete ctx;
}

}  // extern "C"
