// hz_api.cu — the C-ABI entry points of include/hz.h: host-side setup (GLL tables, time-step tables,
// partition, variant choice), the outer DDM driver on one stream, and the launches of the auxiliary
// kernels.  No torch types; device memory of the context is cudaMalloc'd here and freed in hz_destroy.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/hz.h"
#include "hz_aux.cuh"
#include "hz_host_gll.h"
#include "hz_internal.h"
#include "hz_minres.cuh"
#include "hz_quad.cuh"

using namespace hz;

namespace {

std::string g_setup_error;  // message of the last failed hz_mesh_setup (no context exists then)

template <typename T>
cudaError_t dmalloc(T **ptr, size_t n) {
  *ptr = nullptr;
  if (n == 0) return cudaSuccess;
  return cudaMalloc((void **)ptr, n * sizeof(T));
}

inline int roundup(int a, int b) { return (a + b - 1) / b * b; }

struct EventGuard {  // a CUDA event released on scope exit
  cudaEvent_t e = nullptr;
  ~EventGuard() { if (e) cudaEventDestroy(e); }
};

}  // namespace

struct hz_ctx {
  // mesh + physics
  int nx = 0, ny = 0, p = 0, npx = 0, npy = 0, EB = 0;
  double x0 = 0, y0 = 0, x1 = 0, y1 = 0, omega = 0, hx = 0, hy = 0, c_max = 0;
  Gll gll;
  double *d_c = nullptr, *d_fre = nullptr, *d_fim = nullptr, *d_bc = nullptr;
  // general quadrilaterals (hz_mesh_setup_quads): vertex coordinates, the element-wise bound on lmax(M^-1 A)
  // (reading R24), the reference data and, per partition, the geometric factors of every quadrature point
  bool general = false;
  double *d_vx = nullptr, *d_vy = nullptr;
  double lmax_quads = 0;
  RefQ refq{};
  void *d_G = nullptr;
  // partition
  bool part = false;
  int sx = 0, sy = 0, ex = 0, ey = 0, L = 0, E = 0, prec = 0;
  int mx = 0, my = 0, csm = 0, ws = 0, cl = 1, entry = -1, pack = 1;
  int pk = 0;             // the partition launches k_sweep_pack (TileEntry::pk of the chosen entry)
  int cmerge = 0;         // k_sweep_pack: the corner node rides on the last top piece (SweepArgs::cmerge)
  Layout lay{};
  SweepLaunch launch{};
  hz_part_flags flags{};  // variant-choice controls of the last hz_partition_ex
  int worder = 0;         // warp-role order of the warp-specialised kernel
  int n_t = 0;
  double dt = 0, theta = 0, sigma = 0;
  size_t ws_bytes = 0;
  void *d_tab = nullptr, *d_gamma = nullptr, *d_alpha = nullptr, *d_bbf_re = nullptr, *d_bbf_im = nullptr;
  void *d_usub = nullptr, *d_lam = nullptr, *d_g = nullptr, *d_k2 = nullptr, *d_bs = nullptr;
  void *d_bandx = nullptr, *d_bandy = nullptr, *d_scr = nullptr;
  void *d_bbf_zero = nullptr;  // all-zero load of the homogeneous sweep (hz_ddm_solve_mixed), allocated on first use
  void *d_mix = nullptr;       // hz_ddm_solve_mixed: hi context: X_old (n_state doubles); lo context: D (n_state floats)
  double *d_wxl = nullptr, *d_wyl = nullptr;
  int *d_sxp = nullptr, *d_syp = nullptr;           // x / y part of Layout::slot per local node column / row (k_build)
  GatherLine *d_gcol = nullptr, *d_grow = nullptr;  // k_gather's line tables (per global node column / row)
  double *d_part = nullptr, *d_red = nullptr, *d_ures = nullptr;
  void *d_opk2 = nullptr, *d_opy = nullptr;  // hz_operator_time: w^2/c^2 and the output vector, in precision op_prec
  int op_prec = -1;
  int res_blocks = 0;
  Elem1D<double> ex1{}, ey1{};
  // cached CUDA graph of `g_chunk` {sweep, exchange} pairs (use_graph)
  // operator data of the MINRES comparator (built on first use): m | w2M | wH | bf_re | bf_im [L][NS], sedge [L][4][E]
  void *d_mr = nullptr;
  int *d_mr_iters = nullptr;
  double *d_mr_res = nullptr;
  // Krylov workspace of hz_ddm_solve_gmres: kry_vecs vectors of n_state reals; partial sums of the dots
  void *d_kry = nullptr;
  double *d_kpart = nullptr;
  int kry_vecs = 0;
  long long n_state = 0;
  long long kry_len = 0;  // length of the Krylov vectors d_kry was allocated for
  cudaGraphExec_t g_exec = nullptr;
  cudaStream_t cap_stream = nullptr;  // capture happens on this private stream (the legacy default stream cannot capture)
  // hz_ddm_solve_sources: copy-in / copy-out streams, double-buffered staging and the events that order them
  cudaStream_t s_in = nullptr, s_out = nullptr;
  // the boundary-ring kernel of the global operator runs beside the interior kernel on a stream of its own (fork / join by events)
  cudaStream_t s_ring = nullptr;
  cudaEvent_t ev_rfork = nullptr, ev_rjoin = nullptr;
  double *d_fstage[2] = {nullptr, nullptr};
  void *d_ubuf[2] = {nullptr, nullptr};
  size_t ubuf_bytes = 0;
  cudaEvent_t ev_up[2] = {nullptr, nullptr}, ev_build[2] = {nullptr, nullptr}, ev_gather[2] = {nullptr, nullptr},
              ev_down[2] = {nullptr, nullptr};
  int g_chunk = 0, g_nwh = 0, g_warm = 0;
  double g_relax = 0;
  std::vector<double> h_tab;  // host copy of the time-step table (kernel-parameter form of the ws kernel)
  TabC<float> tc32{};
  TabC<double> tc64{};
  std::string err;
};

namespace {

hz_status fail(hz_ctx *ctx, hz_status st, const std::string &msg) {
  if (ctx) ctx->err = msg; else g_setup_error = msg;
  return st;
}
hz_status cuda_fail(hz_ctx *ctx, cudaError_t e, const char *what) {
  return fail(ctx, e == cudaErrorMemoryAllocation ? HZ_ENOMEM : HZ_ECUDA,
              std::string(what) + ": " + cudaGetErrorString(e));
}
#define HZ_CUDA(call)                                        \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); \
  } while (0)

void free_partition(hz_ctx *c) {
  c->d_usub = nullptr;  // lives inside the d_lam allocation (joint state lambda | u_l)
  if (c->d_mr) { cudaFree(c->d_mr); c->d_mr = nullptr; }
  if (c->d_mr_iters) { cudaFree(c->d_mr_iters); c->d_mr_iters = nullptr; }
  if (c->d_mr_res) { cudaFree(c->d_mr_res); c->d_mr_res = nullptr; }
  if (c->d_kry) { cudaFree(c->d_kry); c->d_kry = nullptr; c->kry_vecs = 0; c->kry_len = 0; }
  if (c->d_kpart) { cudaFree(c->d_kpart); c->d_kpart = nullptr; }
  if (c->g_exec) { cudaGraphExecDestroy(c->g_exec); c->g_exec = nullptr; }
  if (c->d_G) { cudaFree(c->d_G); c->d_G = nullptr; }
  void **ptrs[] = {&c->d_tab, &c->d_gamma, &c->d_alpha, &c->d_bbf_re, &c->d_bbf_im, &c->d_lam, &c->d_bbf_zero, &c->d_mix,
                   &c->d_g, &c->d_k2, &c->d_bs, &c->d_bandx, &c->d_bandy, &c->d_scr, (void **)&c->d_wxl, (void **)&c->d_wyl,
                   (void **)&c->d_part, (void **)&c->d_red, (void **)&c->d_ures, (void **)&c->d_gcol, (void **)&c->d_grow, (void **)&c->d_sxp, (void **)&c->d_syp};
  for (void **q : ptrs) { if (*q) cudaFree(*q); *q = nullptr; }
  c->part = false;
  c->ws_bytes = 0;
}

Geo make_geo(const hz_ctx *c) {
  Geo g{};
  g.nx = c->nx; g.ny = c->ny; g.p = c->p; g.npx = c->npx; g.npy = c->npy;
  g.sx = c->sx; g.sy = c->sy; g.ex = c->ex; g.ey = c->ey; g.E = c->E; g.EB = c->EB;
  if (c->sx > 0 && c->sy > 0) {  // (an unpartitioned context: the global kernels do not read these)
    g.exq = c->nx / c->sx; g.exr = c->nx % c->sx; g.eyq = c->ny / c->sy; g.eyr = c->ny % c->sy;
  }
  g.hx = c->hx; g.hy = c->hy; g.omega = c->omega; g.theta = c->theta; g.sigma = c->sigma;
  return g;
}

template <typename real>
hz_status run_build(hz_ctx *ctx, int only_source, cudaStream_t st, const double *f_re = nullptr) {
  if (!f_re) f_re = ctx->d_fre;  // hz_ddm_solve_sources builds from its staging buffers
  const long long total = (long long)ctx->L * ctx->lay.lnx * ctx->lay.lny;
  const int bs = 256;
  const unsigned nb = (unsigned)((total + bs - 1) / bs);
  if (ctx->general) {
    k_build_quad<real><<<nb, bs, 0, st>>>(make_geo(ctx), ctx->lay, ctx->refq, ctx->d_vx, ctx->d_vy, ctx->d_c, f_re,
                                          ctx->d_fim, ctx->d_bc, (real *)ctx->d_gamma, (real *)ctx->d_alpha,
                                          (real *)ctx->d_bbf_re, (real *)ctx->d_bbf_im, (real *)ctx->d_k2,
                                          (real *)ctx->d_bs, only_source);
    HZ_CUDA(cudaGetLastError());
    if (!only_source) {
      const int NQ = (ctx->p + 1) * (ctx->p + 1);
      const long long tq = (long long)ctx->L * ctx->ex * ctx->ey * NQ;
      k_build_quad_metric<real><<<(unsigned)((tq + bs - 1) / bs), bs, 0, st>>>(make_geo(ctx), ctx->refq, ctx->d_vx, ctx->d_vy,
                                                                               ctx->launch.threads, (real *)ctx->d_G);
      HZ_CUDA(cudaGetLastError());
    }
    return HZ_OK;
  }
  auto magic = [](unsigned long long d) { return d <= 1 ? 0ull : ~0ull / d + 1ull; };   // ceil(2^64 / d), d >= 2
  BuildIdx bi{magic((unsigned long long)ctx->lay.lnx * ctx->lay.lny), magic((unsigned long long)ctx->lay.lnx),
              magic((unsigned long long)ctx->sx), ctx->d_sxp, ctx->d_syp};
  k_build<real><<<nb, bs, 0, st>>>(make_geo(ctx), ctx->lay, bi, ctx->d_c, f_re, ctx->d_fim, ctx->d_bc, ctx->d_wxl,
                                   ctx->d_wyl, (real *)ctx->d_gamma, (real *)ctx->d_alpha, (real *)ctx->d_bbf_re,
                                   (real *)ctx->d_bbf_im, (real *)ctx->d_k2, (real *)ctx->d_bs, only_source);
  HZ_CUDA(cudaGetLastError());
  return HZ_OK;
}

template <typename real>
void fill_elem1d(const Gll &g, double h, Elem1D<real> *e) {
  const int P = g.p;
  const double sc = 4.0 / (h * h);
  std::memset(e, 0, sizeof(*e));
  for (int a = 1; a < P; ++a)
    for (int c = 0; c <= P; ++c) e->kin[a][c] = (real)(sc * g.K[a][c] / g.w[a]);
  for (int c = 0; c <= P; ++c) {
    e->k0[c] = (real)(sc * g.K[0][c] / (2.0 * g.w[0]));
    e->kp[c] = (real)(sc * g.K[P][c] / (2.0 * g.w[0]));
  }
}

template <typename real>
cudaError_t upload_as(const std::vector<double> &src, void **dst) {
  std::vector<real> tmp(src.size());
  for (size_t i = 0; i < src.size(); ++i) tmp[i] = (real)src[i];
  cudaError_t e = cudaMalloc(dst, tmp.size() * sizeof(real));
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, tmp.data(), tmp.size() * sizeof(real), cudaMemcpyHostToDevice);
}

template <typename real>
SweepArgs<real> make_args(const hz_ctx *c, const hz_solve_opts *o, bool homog = false) {
  SweepArgs<real> a{};
  a.lay = c->lay;
  a.sx = c->sx; a.sy = c->sy; a.E = c->E;
  a.exq = c->nx / c->sx; a.exr = c->nx % c->sx; a.eyq = c->ny / c->sy; a.eyr = c->ny % c->sy;
  a.n_t = c->n_t; a.n_wh = o->n_wh; a.warm = o->warm_start;
  a.sigma = (real)c->sigma; a.omega = (real)c->omega;
  a.cos_h = (real)std::cos(M_PI / c->n_t); a.sin_h = (real)std::sin(M_PI / c->n_t);
  a.two_over_nt = (real)(2.0 / c->n_t);
  a.tab = (const Tab4<real> *)c->d_tab;
  a.gamma = (const real *)c->d_gamma; a.alpha = (const real *)c->d_alpha;
  a.bbf_re = (const real *)c->d_bbf_re; a.bbf_im = (const real *)c->d_bbf_im;
  if (homog) { a.bbf_re = (const real *)c->d_bbf_zero; a.bbf_im = nullptr; }  // the sweep with the load removed
  a.u_sub = (real *)c->d_usub; a.lam = (const real *)c->d_lam; a.gout = (real *)c->d_g;
  a.k2edge = (const real *)c->d_k2; a.bs = (const real *)c->d_bs;
  a.bandx = (const real *)c->d_bandx; a.bandy = (const real *)c->d_bandy;
  for (int i = 0; i <= kMaxP; ++i) {
    for (int j = 0; j <= kMaxP; ++j) { a.ex1.kin[i][j] = (real)c->ex1.kin[i][j]; a.ey1.kin[i][j] = (real)c->ey1.kin[i][j]; }
    a.ex1.k0[i] = (real)c->ex1.k0[i]; a.ex1.kp[i] = (real)c->ex1.kp[i];
    a.ey1.k0[i] = (real)c->ey1.k0[i]; a.ey1.kp[i] = (real)c->ey1.kp[i];
  }
  a.worder = c->worder;
  a.fused = 0; a.relax = (real)o->relax; a.g_prev = nullptr; a.lam_rw = nullptr;
  a.pack = c->pack; a.L = c->L; a.cmerge = c->cmerge;
  return a;
}

template <typename real>
QuadArgs<real> make_quad_args(const hz_ctx *c) {
  QuadArgs<real> q{};
  q.G = (const real *)c->d_G;
  q.nep = c->launch.threads;
  for (int a = 0; a <= c->p; ++a)
    for (int b = 0; b <= c->p; ++b) q.D[a][b] = (real)c->gll.D[a][b];
  return q;
}

cudaError_t launch_sweep(const hz_ctx *c, const hz_solve_opts *o, cudaStream_t st, bool homog = false) {
  if (c->lay.variant == 3) {
    if (c->prec == HZ_F32)
      return launch_sweep_quad_f32(make_args<float>(c, o, homog), make_quad_args<float>(c), &c->tc32, c->p, c->launch, st);
    return launch_sweep_quad_f64(make_args<double>(c, o, homog), make_quad_args<double>(c), &c->tc64, c->p, c->launch, st);
  }
  if (c->prec == HZ_F32) {
    SweepArgs<float> a = make_args<float>(c, o, homog);
    if (c->lay.variant == 2) return launch_sweep_stream_f32(a, (float *)c->d_scr, c->p, c->launch, st);
    return c->lay.variant == 0 ? launch_sweep_dof_f32(a, c->p, c->launch, st)
                               : launch_sweep_tile_f32(a, &c->tc32, c->entry, c->launch, st);
  }
  SweepArgs<double> a = make_args<double>(c, o, homog);
  if (c->lay.variant == 2) return launch_sweep_stream_f64(a, (double *)c->d_scr, c->p, c->launch, st);
  return c->lay.variant == 0 ? launch_sweep_dof_f64(a, c->p, c->launch, st)
                             : launch_sweep_tile_f64(a, &c->tc64, c->entry, c->launch, st);
}

cudaError_t launch_exchange(const hz_ctx *c, double rho, cudaStream_t st) {
  const long long total = (long long)c->L * 8 * c->E;
  const int bs = 256;
  const unsigned nb = (unsigned)((total + bs - 1) / bs);
  if (c->prec == HZ_F32)
    k_exchange<float><<<nb, bs, 0, st>>>(c->sx, c->sy, c->E, c->lay.lnx, c->lay.lny, (float)rho, (float *)c->d_lam,
                                         (const float *)c->d_g);
  else
    k_exchange<double><<<nb, bs, 0, st>>>(c->sx, c->sy, c->E, c->lay.lnx, c->lay.lny, rho, (double *)c->d_lam,
                                          (const double *)c->d_g);
  return cudaGetLastError();
}

// gather into `out` of type outT (precision prec_out); the line tables are built by hz_partition (upload_gather_tables)
cudaError_t launch_gather(const hz_ctx *c, void *out, int prec_out, cudaStream_t st) {
  const int bs = 256;
  const dim3 grid((unsigned)((c->npx + bs - 1) / bs), (unsigned)c->npy);
  const size_t NS = (size_t)c->lay.NS;
  if (c->prec == HZ_F32) {
    if (prec_out == HZ_F32) k_gather<float, float><<<grid, bs, 0, st>>>(c->npx, c->npy, c->sx, NS, c->d_gcol, c->d_grow, (const float *)c->d_usub, (float *)out);
    else k_gather<float, double><<<grid, bs, 0, st>>>(c->npx, c->npy, c->sx, NS, c->d_gcol, c->d_grow, (const float *)c->d_usub, (double *)out);
  } else {
    if (prec_out == HZ_F32) k_gather<double, float><<<grid, bs, 0, st>>>(c->npx, c->npy, c->sx, NS, c->d_gcol, c->d_grow, (const double *)c->d_usub, (float *)out);
    else k_gather<double, double><<<grid, bs, 0, st>>>(c->npx, c->npy, c->sx, NS, c->d_gcol, c->d_grow, (const double *)c->d_usub, (double *)out);
  }
  return cudaGetLastError();
}

// the per-column / per-row tables of k_gather (hz_aux.cuh): which subdomain(s) hold global node line I (J) and where
cudaError_t upload_gather_tables(hz_ctx *c) {
  const Geo g = make_geo(c);
  auto fill = [&](int np, int n_el, int q, int r, int mul, bool xdir, std::vector<GatherLine> *t) {
    t->resize(np);
    for (int I = 0; I < np; ++I) {
      const int eh = I / g.p > n_el - 1 ? n_el - 1 : I / g.p;
      const int i1 = sub_of_elem(q, r, eh);
      const bool shared = I == sub_off(q, r, i1) * g.p && i1 > 0;
      auto part = [&](int k) {   // x (y) part of Layout::slot of this line in subdomain column (row) k
        const int loc = I - sub_off(q, r, k) * g.p;
        return xdir ? c->lay.slot(loc, 0) : c->lay.slot(0, loc);
      };
      GatherLine L;
      L.s1 = i1 * mul;
      L.p1 = part(i1);
      L.p0 = shared ? part(i1 - 1) : 0;
      L.n = shared ? 2 : 1;
      (*t)[I] = L;
    }
  };
  std::vector<GatherLine> tx, ty;
  fill(c->npx, c->nx, g.exq, g.exr, 1, true, &tx);
  fill(c->npy, c->ny, g.eyq, g.eyr, c->sx, false, &ty);
  cudaError_t e = cudaMalloc((void **)&c->d_gcol, tx.size() * sizeof(GatherLine));
  if (e != cudaSuccess) return e;
  e = cudaMalloc((void **)&c->d_grow, ty.size() * sizeof(GatherLine));
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(c->d_gcol, tx.data(), tx.size() * sizeof(GatherLine), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(c->d_grow, ty.data(), ty.size() * sizeof(GatherLine), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return e;
  // k_build's separable slot tables
  std::vector<int> sxp(c->lay.lnx), syp(c->lay.lny);
  for (int i = 0; i < c->lay.lnx; ++i) sxp[i] = c->lay.slot(i, 0);
  for (int j = 0; j < c->lay.lny; ++j) syp[j] = c->lay.slot(0, j);
  e = cudaMalloc((void **)&c->d_sxp, sxp.size() * sizeof(int));
  if (e != cudaSuccess) return e;
  e = cudaMalloc((void **)&c->d_syp, syp.size() * sizeof(int));
  if (e != cudaSuccess) return e;
  e = cudaMemcpy(c->d_sxp, sxp.data(), sxp.size() * sizeof(int), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return e;
  return cudaMemcpy(c->d_syp, syp.data(), syp.size() * sizeof(int), cudaMemcpyHostToDevice);
}

// launches k_helm<inT, acc, P, MODE> on the whole mesh (hz_aux.cuh)
// overlap_ring: launch the ring kernel on ctx->s_ring, concurrent with the interior kernel (they write disjoint outputs);
// false = both on `st`, nothing created (hz_residual_static)
template <typename inT, typename acc, int MODE>
cudaError_t launch_helm(hz_ctx *ctx, const acc *k2, const void *u_dev, double *part, acc *y, cudaStream_t st, bool overlap_ring = true) {
  HelmC<acc> hc{};
  const int P_ = ctx->p;
  for (int a = 0; a <= P_; ++a) {
    hc.w[a] = (acc)ctx->gll.w[a];
    hc.wa[a] = (acc)(a == 0 ? ctx->gll.w[0] + ctx->gll.w[P_] : ctx->gll.w[a]);
    for (int b = 0; b <= P_; ++b) {
      hc.kx[a][b] = (acc)(ctx->hy / ctx->hx * ctx->gll.K[a][b]);
      hc.ky[a][b] = (acc)(ctx->hx / ctx->hy * ctx->gll.K[a][b]);
    }
  }
  hc.mh = (acc)(0.25 * ctx->hx * ctx->hy);
  for (int cc = -P_; cc <= P_; ++cc) {   // assembled row of a node shared by two elements
    const double kl = cc <= 0 ? ctx->gll.K[P_][cc + P_] : 0.0, kr = cc >= 0 ? ctx->gll.K[0][cc] : 0.0;
    hc.kx0[cc + P_] = (acc)(ctx->hy / ctx->hx * (kl + kr));
    hc.ky0[cc + P_] = (acc)(ctx->hx / ctx->hy * (kl + kr));
  }
  for (int b = 0; b < P_; ++b)
    for (int a = 0; a < P_; ++a) {
      const double wa_ = a == 0 ? ctx->gll.w[0] + ctx->gll.w[P_] : ctx->gll.w[a], wb_ = b == 0 ? ctx->gll.w[0] + ctx->gll.w[P_] : ctx->gll.w[b];
      hc.wm[b][a] = (acc)(0.25 * ctx->hx * ctx->hy * wa_ * wb_);
    }
  const Geo g = make_geo(ctx);
  const HelmGrid hg = helm_grid(ctx->nx, ctx->ny, ctx->p);
  const dim3 block(kHelmBX, kHelmBY);
  const size_t sm = helm_smem(ctx->p, sizeof(inT), MODE == 1 ? sizeof(acc) : 0);
  using fe_t = void (*)(Geo, const HelmGrid, const HelmC<acc>, const double *, const acc *, const double *, const double *,
                        const double *, const inT *, double *, acc *);
  using ft_t = void (*)(Geo, const HelmGrid, const HelmC<acc>, const double *, const acc *, const double *, const double *,
                        const inT *, double *, acc *);
  fe_t fi = nullptr;   // patches strictly inside the mesh, cp.async staging
  ft_t ft = nullptr;   // the same with TMA bulk-copy staging: the fp64 operator at P >= 3 (hz_aux.cuh)
  fe_t fe = nullptr;   // the ring of patches that touch the mesh boundary
  constexpr bool kTma = MODE == 1 && sizeof(inT) == 8;
  switch (ctx->p) {
    case 1: fi = k_helm<inT, acc, 1, MODE, false>; fe = k_helm<inT, acc, 1, MODE, true>; break;
    case 2: fi = k_helm<inT, acc, 2, MODE, false>; fe = k_helm<inT, acc, 2, MODE, true>; break;
    case 3: fi = k_helm<inT, acc, 3, MODE, false>; fe = k_helm<inT, acc, 3, MODE, true>; if constexpr (kTma) ft = k_helm_tma<inT, acc, 3, 1>; break;
    case 4: fi = k_helm<inT, acc, 4, MODE, false>; fe = k_helm<inT, acc, 4, MODE, true>; if constexpr (kTma) ft = k_helm_tma<inT, acc, 4, 1>; break;
    default: return cudaErrorInvalidValue;
  }
  const size_t smt = helm_tma_smem(ctx->p, sizeof(inT), sizeof(acc));
  cudaError_t e = cudaFuncSetAttribute(fi, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(fe, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
  if (e != cudaSuccess) return e;
  if (ft) {
    e = cudaFuncSetAttribute(ft, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smt);
    if (e != cudaSuccess) return e;
  }
  const int nix = hg.bxh - 1, niy = hg.byh - 1, nring = hg.gx * hg.gy - nix * niy;
  const bool both = nix > 0 && niy > 0 && nring > 0;
  cudaStream_t sr = st;
  if (both && overlap_ring) {
    if (!ctx->s_ring) {
      e = cudaStreamCreateWithFlags(&ctx->s_ring, cudaStreamNonBlocking);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_rfork, cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_rjoin, cudaEventDisableTiming);
      if (e != cudaSuccess) return e;
    }
    e = cudaEventRecord(ctx->ev_rfork, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->s_ring, ctx->ev_rfork, 0);
    if (e != cudaSuccess) return e;
    sr = ctx->s_ring;
  }
  if (nring > 0)
    fe<<<dim3(nring), block, sm, sr>>>(g, hg, hc, ctx->d_c, k2, ctx->d_fre, ctx->d_fim, ctx->d_bc, (const inT *)u_dev, part, y);
  if (nix > 0 && niy > 0) {
    if (ft) ft<<<dim3(nix, niy), block, smt, st>>>(g, hg, hc, ctx->d_c, k2, ctx->d_fre, ctx->d_fim, (const inT *)u_dev, part, y);
    else fi<<<dim3(nix, niy), block, sm, st>>>(g, hg, hc, ctx->d_c, k2, ctx->d_fre, ctx->d_fim, ctx->d_bc, (const inT *)u_dev, part, y);
  }
  if (sr != st) {
    e = cudaEventRecord(ctx->ev_rjoin, sr);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ctx->ev_rjoin, 0);
    if (e != cudaSuccess) return e;
  }
  return cudaGetLastError();
}

hz_status residual_impl(hz_ctx *ctx, const void *u_dev, int u_prec, double *rel, cudaStream_t st) {
  const long long total = (long long)ctx->npx * ctx->npy;
  const int bs = 256;
  const int nb = ctx->general ? (int)((total + bs - 1) / bs)
                              : ((ctx->nx + 1 + kHelmBX - 1) / kHelmBX) * ((ctx->ny + 1 + kHelmBY - 1) / kHelmBY);
  if (!ctx->d_part || ctx->res_blocks != nb) {
    if (ctx->d_part) cudaFree(ctx->d_part);
    if (ctx->d_red) cudaFree(ctx->d_red);
    ctx->d_part = nullptr; ctx->d_red = nullptr;
    HZ_CUDA(dmalloc(&ctx->d_part, (size_t)2 * nb));
    HZ_CUDA(dmalloc(&ctx->d_red, 2));
    ctx->res_blocks = nb;
  }
  if (ctx->general) {
    Geo g = make_geo(ctx);
    if (u_prec == HZ_F32)
      k_residual_quad<float><<<nb, bs, 0, st>>>(g, ctx->refq, ctx->d_vx, ctx->d_vy, ctx->d_c, ctx->d_fre, ctx->d_fim,
                                                ctx->d_bc, (const float *)u_dev, ctx->d_part);
    else
      k_residual_quad<double><<<nb, bs, 0, st>>>(g, ctx->refq, ctx->d_vx, ctx->d_vy, ctx->d_c, ctx->d_fre, ctx->d_fim,
                                                 ctx->d_bc, (const double *)u_dev, ctx->d_part);
    HZ_CUDA(cudaGetLastError());
  } else if (u_prec == HZ_F32) {
    HZ_CUDA((launch_helm<float, double, 0>(ctx, nullptr, u_dev, ctx->d_part, nullptr, st)));
  } else {
    HZ_CUDA((launch_helm<double, double, 0>(ctx, nullptr, u_dev, ctx->d_part, nullptr, st)));
  }
  k_reduce2<<<1, 1024, 0, st>>>(ctx->d_part, nb, ctx->d_red);
  HZ_CUDA(cudaGetLastError());
  double h[2];
  HZ_CUDA(cudaMemcpyAsync(h, ctx->d_red, sizeof(h), cudaMemcpyDeviceToHost, st));
  HZ_CUDA(cudaStreamSynchronize(st));
  *rel = (h[1] > 0.0) ? std::sqrt(h[0] / h[1]) : std::sqrt(h[0]);
  return HZ_OK;
}

// Can the device co-schedule one cluster of t.cl CTAs of this shape at all?  (cudaOccupancyMaxActiveClusters; an
// unschedulable cluster would otherwise only surface as a launch error.)  Errors count as "no".
bool cluster_schedulable(const TileEntry &t, const SweepLaunch &la) {
  if (cudaFuncSetAttribute(t.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)la.smem) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  if (t.cl > 8 && cudaFuncSetAttribute(t.fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3(la.blocks, 1, 1);
  lc.blockDim = dim3(la.threads, 1, 1);
  lc.dynamicSmemBytes = la.smem;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = t.cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  lc.attrs = at; lc.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, t.fn, &lc) != cudaSuccess) { cudaGetLastError(); return false; }
  return n > 0;
}

}  // namespace

extern "C" {

hz_status hz_mesh_setup(hz_ctx **out, int nx, int ny, double x0, double y0, double x1, double y1, int p,
                        const double *c_nodes, double omega, const double *f_re, const double *f_im,
                        const double *bc_lambda) {
  hz_ctx *ctx = nullptr;  // for the HZ_CUDA macro before the context exists
  if (!out || !c_nodes || !f_re) return fail(nullptr, HZ_EINVAL, "hz_mesh_setup: NULL out, c_nodes or f_re");
  if (nx < 1 || ny < 1 || !(x1 > x0) || !(y1 > y0) || !(omega > 0.0) || !std::isfinite(omega))
    return fail(nullptr, HZ_EINVAL, "hz_mesh_setup: need nx,ny >= 1, x1 > x0, y1 > y0, omega > 0");
  if (p < 1 || p > kMaxP) return fail(nullptr, HZ_EUNSUPPORTED, "hz_mesh_setup: degree p must be 1..4");
  const long long nn = ((long long)nx * p + 1) * ((long long)ny * p + 1);
  if (nn > (1ll << 31) - 1) return fail(nullptr, HZ_EUNSUPPORTED, "hz_mesh_setup: more than 2^31-1 nodes");
  double cmax = 0.0;
  for (long long q = 0; q < nn; ++q) {
    if (!(c_nodes[q] > 0.0) || !std::isfinite(c_nodes[q])) return fail(nullptr, HZ_EINVAL, "hz_mesh_setup: c_nodes must be finite and > 0");
    cmax = std::fmax(cmax, c_nodes[q]);
  }
  hz_ctx *c = new (std::nothrow) hz_ctx();
  if (!c) return fail(nullptr, HZ_ENOMEM, "hz_mesh_setup: out of host memory");
  c->nx = nx; c->ny = ny; c->p = p; c->npx = nx * p + 1; c->npy = ny * p + 1;
  c->EB = c->npx > c->npy ? c->npx : c->npy;
  c->x0 = x0; c->y0 = y0; c->x1 = x1; c->y1 = y1; c->omega = omega;
  c->hx = (x1 - x0) / nx; c->hy = (y1 - y0) / ny; c->c_max = cmax;
  make_gll(p, &c->gll);
  cudaError_t e = cudaSuccess;
  const size_t bytes = (size_t)nn * sizeof(double);
  if (e == cudaSuccess) e = dmalloc(&c->d_c, (size_t)nn);
  if (e == cudaSuccess) e = dmalloc(&c->d_fre, (size_t)nn);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_c, c_nodes, bytes, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_fre, f_re, bytes, cudaMemcpyHostToDevice);
  if (e == cudaSuccess && f_im) {
    e = dmalloc(&c->d_fim, (size_t)nn);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_fim, f_im, bytes, cudaMemcpyHostToDevice);
  }
  if (e == cudaSuccess && bc_lambda) {
    e = dmalloc(&c->d_bc, (size_t)8 * c->EB);
    if (e == cudaSuccess) e = cudaMemcpy(c->d_bc, bc_lambda, (size_t)8 * c->EB * sizeof(double), cudaMemcpyHostToDevice);
  }
  if (e != cudaSuccess) {
    hz_status st = cuda_fail(nullptr, e, "hz_mesh_setup (device allocation / copy)");
    hz_destroy(c);
    return st;
  }
  (void)ctx;
  *out = c;
  return HZ_OK;
}

hz_status hz_mesh_setup_quads(hz_ctx **out, int nx, int ny, int p, const double *vx, const double *vy,
                              const double *c_nodes, double omega, const double *f_re, const double *f_im,
                              const double *bc_lambda) {
  if (!vx || !vy) return fail(nullptr, HZ_EINVAL, "hz_mesh_setup_quads: NULL vertex arrays");
  if (nx < 1 || ny < 1 || p < 1 || p > kMaxP || !out || !c_nodes)
    return hz_mesh_setup(out, nx, ny, 0.0, 0.0, 1.0, 1.0, p, c_nodes, omega, f_re, f_im, bc_lambda);  // its messages
  // element-wise bound on lmax(M^-1 A) (reading R24):  Lhat (Gx + Gy) / mu  with  Lhat = Lambda_p / 4,
  // Gx = max_q (gxx + |gxy|), Gy = max_q (gyy + |gxy|), mu = min_q detJ / c^2 over the element's GLL points
  Gll gl;
  make_gll(p, &gl);
  const int npx = nx * p + 1;
  double lmax = 0.0;
  for (int gy = 0; gy < ny; ++gy)
    for (int gx = 0; gx < nx; ++gx) {
      double X[4], Y[4];
      quad_vertices(vx, vy, nx, gx, gy, X, Y);
      double Gx = 0.0, Gy = 0.0, mu = INFINITY;
      for (int b = 0; b <= p; ++b)
        for (int a = 0; a <= p; ++a) {
          const QuadPt q = quad_point(X, Y, gl.xi[a], gl.xi[b]);
          if (!(q.det > 0.0) || !std::isfinite(q.det))
            return fail(nullptr, HZ_EINVAL, "hz_mesh_setup_quads: an element is not convex / not counter-clockwise");
          const double cc = c_nodes[(size_t)(gy * p + b) * npx + gx * p + a];
          Gx = std::fmax(Gx, q.gxx + std::fabs(q.gxy));
          Gy = std::fmax(Gy, q.gyy + std::fabs(q.gxy));
          mu = std::fmin(mu, q.det / (cc * cc));
        }
      lmax = std::fmax(lmax, 0.25 * gl.lambda_p * (Gx + Gy) / mu);
    }
  hz_ctx *c = nullptr;
  // hx = hy = 1 in the rectangular fields: unused by the general-geometry kernels
  hz_status stt = hz_mesh_setup(&c, nx, ny, 0.0, 0.0, (double)nx, (double)ny, p, c_nodes, omega, f_re, f_im, bc_lambda);
  if (stt != HZ_OK) return stt;
  c->general = true;
  c->lmax_quads = lmax;
  for (int a = 0; a <= p; ++a) {
    c->refq.xi[a] = gl.xi[a]; c->refq.w[a] = gl.w[a];
    for (int b = 0; b <= p; ++b) c->refq.D[a][b] = gl.D[a][b];
  }
  const size_t nv = (size_t)(nx + 1) * (ny + 1);
  cudaError_t e = dmalloc(&c->d_vx, nv);
  if (e == cudaSuccess) e = dmalloc(&c->d_vy, nv);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_vx, vx, nv * sizeof(double), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_vy, vy, nv * sizeof(double), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    hz_status st2 = cuda_fail(nullptr, e, "hz_mesh_setup_quads (device allocation / copy)");
    hz_destroy(c);
    return st2;
  }
  *out = c;
  return HZ_OK;
}

hz_status hz_set_source(hz_ctx *ctx, const double *f_re, const double *f_im) {
  if (!ctx) return HZ_EINVAL;
  if (!f_re) return fail(ctx, HZ_EINVAL, "hz_set_source: NULL f_re");
  const size_t nn = (size_t)ctx->npx * ctx->npy;
  if (f_im && !ctx->d_fim) {
    if (ctx->part && (ctx->lay.variant == 1))
      return fail(ctx, HZ_EUNSUPPORTED, "hz_set_source: complex f needs the one-DOF-per-thread variant; re-partition");
    HZ_CUDA(dmalloc(&ctx->d_fim, nn));
    // the cached CUDA graph captured kernels whose arguments hold bbf_im == NULL: it must not be replayed
    if (ctx->g_exec) { cudaGraphExecDestroy(ctx->g_exec); ctx->g_exec = nullptr; ctx->g_chunk = 0; }
    if (ctx->part && !ctx->d_bbf_im) {
      const size_t rs = ctx->prec == HZ_F32 ? 4 : 8;
      HZ_CUDA(cudaMalloc(&ctx->d_bbf_im, (size_t)ctx->L * ctx->lay.NS * rs));
      HZ_CUDA(cudaMemset(ctx->d_bbf_im, 0, (size_t)ctx->L * ctx->lay.NS * rs));
    }
  }
  HZ_CUDA(cudaMemcpyAsync(ctx->d_fre, f_re, nn * sizeof(double), cudaMemcpyHostToDevice, 0));
  if (f_im) HZ_CUDA(cudaMemcpyAsync(ctx->d_fim, f_im, nn * sizeof(double), cudaMemcpyHostToDevice, 0));
  else if (ctx->d_fim) HZ_CUDA(cudaMemsetAsync(ctx->d_fim, 0, nn * sizeof(double), 0));
  if (ctx->part) {
    hz_status st = ctx->prec == HZ_F32 ? run_build<float>(ctx, 1, 0) : run_build<double>(ctx, 1, 0);
    if (st != HZ_OK) return st;
  }
  HZ_CUDA(cudaStreamSynchronize(0));
  return HZ_OK;
}

hz_status hz_partition(hz_ctx *ctx, int sx, int sy, hz_transmission tc, hz_prec prec, int dofs_per_thread,
                       double cfl_frac, hz_part_info *info_out) {
  return hz_partition_ex(ctx, sx, sy, tc, prec, dofs_per_thread, cfl_frac, nullptr, info_out);
}

hz_status hz_partition_ex(hz_ctx *ctx, int sx, int sy, hz_transmission tc, hz_prec prec, int dofs_per_thread,
                          double cfl_frac, const hz_part_flags *flags, hz_part_info *info_out) {
  if (!ctx) return HZ_EINVAL;
  hz_part_flags fl{};
  if (flags) fl = *flags;
  if (fl.cluster < -1 || fl.cluster == 1 || fl.grid_blocks < 0 || fl.warp_order < 0 || fl.warp_order > 3 || fl.pack < 0)
    return fail(ctx, HZ_EINVAL, "hz_partition_ex: bad flags");
  if (sx < 1 || sy < 1 || sx > ctx->nx || sy > ctx->ny)
    return fail(ctx, HZ_EINVAL, "hz_partition: need 1 <= sx <= nx, 1 <= sy <= ny");
  if (!ctx->general && (ctx->nx % sx || ctx->ny % sy))
    return fail(ctx, HZ_EINVAL, "hz_partition: sx, sy must divide nx, ny on a uniform mesh (ragged partitions: hz_mesh_setup_quads)");
  if (tc != HZ_TC_IMPEDANCE0) return fail(ctx, HZ_EUNSUPPORTED, "hz_partition: only HZ_TC_IMPEDANCE0");
  if (prec != HZ_F32 && prec != HZ_F64) return fail(ctx, HZ_EINVAL, "hz_partition: bad precision");
  if (!(cfl_frac > 0.0) || cfl_frac > 1.0) return fail(ctx, HZ_EINVAL, "hz_partition: cfl_frac must be in (0,1]");
  if (dofs_per_thread < -1) return fail(ctx, HZ_EINVAL, "hz_partition: dofs_per_thread < -1");
  free_partition(ctx);
  ctx->flags = fl;
  ctx->worder = 0;
  ctx->pack = 1;
  ctx->pk = 0;
  ctx->cmerge = 0;
  const int P = ctx->p;
  // ex, ey: elements per subdomain side; for a ragged partition (general quads only, reading R25) the maximum
  ctx->sx = sx; ctx->sy = sy; ctx->ex = (ctx->nx + sx - 1) / sx; ctx->ey = (ctx->ny + sy - 1) / sy;
  ctx->L = sx * sy; ctx->prec = prec;
  const int lnx = ctx->ex * P + 1, lny = ctx->ey * P + 1, N = lnx * lny;
  ctx->E = lnx > lny ? lnx : lny;
  const size_t rs = prec == HZ_F32 ? 4 : 8;

  // --- time step (reading R9): dt_stab = 2 / sqrt(c_max^2 Lambda_p (1/hx^2 + 1/hy^2)) ---
  const double lmax = ctx->general ? ctx->lmax_quads  // reading R24: element-wise form of the same bound
                                   : ctx->c_max * ctx->c_max * ctx->gll.lambda_p * (1.0 / (ctx->hx * ctx->hx) + 1.0 / (ctx->hy * ctx->hy));
  const double dt_stab = 2.0 / std::sqrt(lmax);
  const double T = 2.0 * M_PI / ctx->omega;
  int n_t = (int)std::ceil(T / (cfl_frac * dt_stab) * (1.0 - 1e-12));
  if (n_t < 4) n_t = 4;
  ctx->n_t = n_t;
  ctx->dt = T / n_t;
  ctx->theta = std::tan(ctx->omega * ctx->dt / 2.0) / ctx->omega;
  ctx->sigma = std::sin(ctx->omega * ctx->dt / 2.0) / (ctx->omega / 2.0);

  // --- variant choice ---
  const TileEntry *tiles = nullptr;
  const int ntiles = prec == HZ_F32 ? tile_table_f32(&tiles) : tile_table_f64(&tiles);
  const size_t tab_bytes = (size_t)n_t * 4 * rs;
  const size_t smem_cap = 227 * 1024;
  Layout lay{};
  lay.lnx = lnx; lay.lny = lny;
  int best = -1, bpack = 1, bcm = 0;
  SweepLaunch bl{};
  Layout blay{};
  int sm_count = 148, dev = 0;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
  const bool no_ws = fl.no_warp_spec != 0, no_cl = fl.cluster == -1, no_regcap = fl.no_reg_cap != 0;
  const int force_cl = fl.cluster > 1 ? fl.cluster : 0;
  const long long Lsel = fl.grid_blocks > 0 ? fl.grid_blocks : (long long)sx * sy;  // grid size the choice assumes
  auto tile_fit = [&](const TileEntry &t, Layout *lo, SweepLaunch *la, int *gsel, int *cmsel) -> bool {
    if (t.p != P || ctx->ex % t.mx || ctx->ey % t.my) return false;
    if (force_cl > 1 && t.cl != force_cl) return false;
    if (fl.pack > 1 && !t.pk) return false;
    Layout q = lay;
    q.variant = 1; q.TX = t.mx * P; q.TY = t.my * P;
    q.cm = t.cl > 1 ? 1 : 0;
    q.ntx = ctx->ex / t.mx + 1; q.nty = ctx->ey / t.my + 1;
    const int ntv = roundup(q.ntx * q.nty, 32);   // virtual tile slots (stride of the per-node arrays)
    int nthr = ntv, ntv_pack = 0;
    size_t sm = 0;
    const size_t narr = 2 * (size_t)(q.TX + q.TY);
    int G = 1;
    if (t.pk) {
      // G subdomains per block: the G*NB full tiles fill whole bulk warps (hz_sweep_pack.cuh)
      // corner node on the last top piece's lane (one edge piece fewer per subdomain) or as a piece of its own: measured per
      // shape on config 5 (A/B on one box, round 2): merging wins for the two-subdomain and 16x16-tile entries, in fp32 for the
      // 1-tile subdomains and at p = 4 (22.4 against 26.4 ms), in fp64 everywhere except p = 3 (50.0 against 47.0 ms); it loses
      // in fp32 at p = 1, 2 with 16 tiles (15.5 against 12.1 ms, 19.2 against 16.2 ms)
      const int NB = (q.ntx - 1) * (q.nty - 1);
      const bool cmerge = t.pk >= 3 || (rs == 4 ? (NB == 1 || P == 4) : P != 3);
      const int NE = q.ntx + q.nty - (cmerge ? 2 : 1);
      if (n_t > kTabCMax) return false;
      if (fl.pack == 1) return false;
      // pk = 3: TWO subdomains of up to 64 full tiles per block, their 2 x (ntx + nty - 2) <= 32 edge pieces in ONE edge
      // warp (the headline shape: 8 x 8 tiles); only when the grid still fills the register-capped occupancy
      // pk = 4: ONE larger subdomain per block through the same kernel (the corner node on the last top piece: 32 edge
      // pieces = one edge warp at 16 x 16 tiles, where k_sweep_ws needs two)
      const bool pair = t.pk == 3, single = t.pk == 4;
      if (pair) {
        if (NB <= 16 || NB > 64 || 2 * NE > 32 || (fl.pack > 1 && fl.pack != 2)) return false;
        if (t.ntx > 0 && (q.ntx != t.ntx || q.nty != t.ntx)) return false;   // compiled for that tile grid
        if (fl.pack == 0 && (Lsel + 1) / 2 < (long long)sm_count * t.minb) return false;
      } else if (single) {
        if (NB <= 64 || fl.pack > 1) return false;
        if (t.ntx > 0 && (q.ntx != t.ntx || q.nty != t.ntx)) return false;
      } else {
        if (NB > 16) return false;   // packing several subdomains per warp only pays below one warp of full tiles
        // own part of a step before (pk = 2) or after (pk = 1) the block barrier: measured per shape on config 5
        // (hz_sweep_pack.cuh, profiles/r02_config_sweep.md)
        const bool pre = NB < 16 || t.mx == 1 || (rs == 8 && P == 1);
        if ((t.pk == 2) != pre) return false;
      }
      auto gcd = [](int a, int b) { while (b) { const int r = a % b; a = b; b = r; } return a; };
      const size_t v16 = 16 / rs;
      const size_t chx = ((size_t)q.TX + v16 - 1) / v16 * v16, chy = ((size_t)q.TY + v16 - 1) / v16 * v16;
      const size_t rsw = 2 * chx + 2 * chy + v16;  // square tiles: 4 chunks + 16 bytes
      const size_t nep = ((size_t)NE + 1 + v16 - 1) / v16 * v16;
      auto shape = [&](int g, int *thr, size_t *smb) {
        *thr = roundup(g * NB, 32) + roundup(g * NE, 32);
        // per buffer: g slices of (padded record grid + zero record + PA | RA) and the scratch region of the idle lanes
        const bool pad = t.ntx > 0;   // compile-time tile grid: padded record grid (hz_sweep_pack.cuh)
        const size_t nrec = pad ? (size_t)(q.ntx + 1) * (q.nty + 1) : (size_t)q.ntx * q.nty, nscr = pad ? 2 * (size_t)(q.ntx + 1) + 3 : 1;
        *smb = 2 * ((size_t)g * ((nrec + 1) * rsw + 2 * nep) + nscr * rsw) * rs;
      };
      if (pair || single) {
        G = pair ? 2 : 1;
      } else if (fl.pack > 1) {
        G = fl.pack;
      } else {
        G = 32 / gcd(32, NB);                        // smallest G that fills the bulk warps ...
        // ... and for 16-tile subdomains four bulk warps (measured on config 5, profiles/r02_config_sweep.md: p = 4,
        // side 4: 8.75 -> 6.77 ms from G = 2 to 8; 4-tile subdomains are faster with one bulk warp than with two)
        if (NB == 16) G = 8;
        for (;; G /= 2) {
          int t2; size_t s2;
          shape(G, &t2, &s2);
          if ((t2 <= t.maxt && s2 <= smem_cap) || G == 1) break;
        }
        // a small grid keeps its parallelism: at least two blocks per SM before subdomains share a block
        while (G > 1 && (Lsel + G - 1) / G < 2LL * sm_count) G /= 2;
        for (;; G /= 2) {
          shape(G, &nthr, &sm);
          if ((nthr <= t.maxt && sm <= smem_cap) || G == 1) break;
        }
      }
      shape(G, &nthr, &sm);
      if (G < 2 && !single) return false;
      ntv_pack = q.ntx * q.nty;
    } else if (t.cl > 1 && t.ws) {
      // cluster kernel with warp-specialised edge pieces (hz_sweep_cw.cuh): the full-tile columns are cut into t.cl strips
      if (no_cl || n_t > kTabCMax || q.ntx - 1 < t.cl) return false;
      const int nbc = q.ntx - 1, nbr = q.nty - 1, wmax = (nbc + t.cl - 1) / t.cl, nel = nbr + wmax + 1;
      nthr = roundup(wmax * nbr, 32) + roundup(nel, 32);
      const size_t v16 = 16 / rs;
      const size_t chx = ((size_t)q.TX + v16 - 1) / v16 * v16, chy = ((size_t)q.TY + v16 - 1) / v16 * v16;
      size_t rsw = 2 * chx + 2 * chy;
      if ((rsw / v16) % 2 == 0) rsw += v16;
      const size_t nep = ((size_t)nel + v16 - 1) / v16 * v16;
      // per buffer: the padded record grid (wmax + 2) x (nty + 1) + the scratch region of the idle lanes + PA | RA; the scalar halo slots of the top pieces
      const size_t bufw = ((size_t)(wmax + 2) * (q.nty + 1) + 2 * (size_t)(q.nty + 1) + 1) * rsw + 2 * nep, hs = 2 * v16;
      sm = (2 * bufw + 2 * hs) * rs + 16;
    } else if (t.cl > 1) {
      if (no_cl || n_t > kTabCMax || q.ntx < t.cl) return false;
      const int wmax = (q.ntx + t.cl - 1) / t.cl;
      nthr = roundup(wmax * q.nty, 32);
      const size_t v16 = 16 / rs;
      const size_t chx = ((size_t)q.TX + v16 - 1) / v16 * v16, chy = ((size_t)q.TY + v16 - 1) / v16 * v16;
      size_t rsw = 2 * chx + 2 * chy;
      if ((rsw / v16) % 2 == 0) rsw += v16;
      sm = 2 * (size_t)(nthr + 33) * rsw * rs + 2 * (size_t)(2 * q.nty) * chy * rs + 16;  // records, halo slots, 2 mbarriers
    } else if (t.ws) {
      if (no_ws || n_t > kTabCMax) return false;
      nthr = roundup((q.ntx - 1) * (q.nty - 1), 32) + roundup(q.ntx + q.nty - 1, 32);
      const int nbulk = (q.ntx - 1) * (q.nty - 1), nedge = q.ntx + q.nty - 1;
      const size_t nrec = (size_t)ntv + 64;
      const size_t v16 = 16 / rs, chx = ((size_t)q.TX + v16 - 1) / v16 * v16;  // chunk length (square tiles)
      sm = 2 * (nrec * (4 * chx + v16) + 2 * (size_t)roundup(nedge, 32)) * rs + (t.csm ? 2 * (size_t)q.TX * q.TY * nthr * rs : 0);
    } else {
      if (n_t > kTabCMax) return false;
      const size_t v16 = 16 / rs;
      const size_t chx = ((size_t)q.TX + v16 - 1) / v16 * v16, chy = ((size_t)q.TY + v16 - 1) / v16 * v16;
      size_t rsw = 2 * chx + 2 * chy;                       // record stride, odd number of 16-byte units
      if ((rsw / v16) % 2 == 0) rsw += v16;
      size_t cst = (2 * (size_t)q.TX * q.TY + v16 - 1) / v16 * v16;  // CSM strip per thread
      if ((cst / v16) % 2 == 0) cst += v16;
      sm = 2 * (size_t)(nthr + 33) * rsw * rs + (t.csm ? (size_t)nthr * cst * rs : 0);
    }
    if (nthr > t.maxt) return false;
    q.NT = t.pk ? ntv_pack : ntv; q.NS = q.TX * q.TY * q.NT;
    if (sm > smem_cap) return false;
    *lo = q; la->blocks = t.pk ? (ctx->L + G - 1) / G : ctx->L * t.cl; la->threads = nthr; la->smem = sm;
    if (gsel) *gsel = G;
    if (cmsel) *cmsel = t.pk ? ((t.pk >= 3 || (rs == 4 ? ((q.ntx - 1) * (q.nty - 1) == 1 || P == 4) : P != 3)) ? 1 : 0) : 0;
    if (t.cl > 1 && !cluster_schedulable(t, *la)) return false;  // e.g. a GPC that cannot co-schedule t.cl such CTAs
    return true;
  };
  const bool complex_f = ctx->d_fim != nullptr;
  bool streamed = dofs_per_thread == -1;
  bool quad = false;
  if (ctx->general) {  // one thread per element, the element's nodes in registers (hz_sweep_quad.cuh)
    if (dofs_per_thread != 0)
      return fail(ctx, HZ_EUNSUPPORTED, "hz_partition: general quadrilaterals have one variant; pass dofs_per_thread = 0");
    const int ne = ctx->ex * ctx->ey;
    if (ne > 1024) return fail(ctx, HZ_EUNSUPPORTED, "hz_partition: general quadrilaterals need <= 1024 elements per subdomain");
    const int n1 = P + 1, v16 = (int)(16 / rs);
    const int ch = roundup(n1, v16);
    int rsw = 4 * ch;
    if ((rsw / v16) % 2 == 0) rsw += v16;
    int cst = n1 * (4 * n1 + roundup(3 * n1, v16));
    if ((cst / v16) % 2 == 0) cst += v16;
    const int nthr = roundup(ne, 32);
    const size_t sm = (2 * (size_t)(nthr + 2) * rsw + (size_t)nthr * cst) * rs;
    if (sm > smem_cap) return fail(ctx, HZ_EUNSUPPORTED, "hz_partition: general quadrilaterals: the subdomain does not fit the shared memory of one SM");
    lay.variant = 3; lay.TX = lay.TY = P; lay.ntx = ctx->ex; lay.nty = ctx->ey; lay.NT = nthr; lay.NS = roundup(N, 32);
    ctx->lay = lay; ctx->mx = ctx->my = 1; ctx->csm = 1; ctx->ws = 0; ctx->cl = 1;
    ctx->launch.blocks = ctx->L; ctx->launch.threads = nthr; ctx->launch.smem = sm;
    quad = true;
  } else if (streamed) {
  } else if (dofs_per_thread == 1 || (dofs_per_thread == 0 && complex_f)) {
    if (N > 1024) {
      if (dofs_per_thread == 1) return fail(ctx, HZ_EUNSUPPORTED, "hz_partition: one DOF per thread needs <= 1024 DOFs per subdomain");
      streamed = true;
    }
  } else {
    for (int i = 0; i < ntiles; ++i) {
      const TileEntry &t = tiles[i];
      const int k = t.mx * P * t.my * P;
      if (dofs_per_thread > 1 && k != dofs_per_thread) continue;
      Layout lo; SweepLaunch la;
      int gsel = 1, cmsel = 0;
      if (!tile_fit(t, &lo, &la, &gsel, &cmsel)) continue;
      // prefer the warp-specialised kernel, then register-resident coefficients, then the smaller tile
      // (more threads, better latency hiding); among otherwise equal instantiations take the
      // register-capped one (higher occupancy, a few spills) only when the grid can fill that occupancy
      if (t.minb > 1 && (Lsel < (long long)sm_count * t.minb || no_regcap)) continue;
      auto score_of = [&](const TileEntry &q) {
        const long long k_ = (long long)q.mx * P * q.my * P;
        // register-resident coefficients first; there the warp-specialised kernel wins and tiles of 9..16 DOFs
        // per thread are the sweet spot (smaller tiles exchange too much, larger ones leave too few warps);
        // with shared-memory coefficients (large subdomains, one block per SM) the smaller tile wins
        const long long nbulk_ = (long long)(ctx->ex / q.mx) * (ctx->ey / q.my);
        // ... provided the subdomain still has two warps of full tiles; otherwise the smaller tile
        const long long dk = nbulk_ < 64 ? 100 + k_ : (k_ < 9 ? 9 - k_ : (k_ > 16 ? k_ - 16 : 0));
        // tiers: (0) one CTA, everything in registers; (1) one CTA, warp-specialised, coefficients in shared memory,
        // tiles of at most 16 DOFs; (2) clusters, smallest first; (3) the remaining shared-memory-coefficient kernels
        // (measured order on configs 4 and 5, profiles/r01_config_sweep.md)
        // (-1) several small subdomains per block, whenever a subdomain has at most 16 full tiles; largest tile <= 16 DOFs
        // fp32: the largest tile; fp64 (16-DOF tiles spill): the tile that gives a subdomain closest to 16 full tiles
        if (q.pk) return -1000000000LL + (rs == 8 ? 100 * std::llabs(nbulk_ - 16) + k_ : (k_ <= 16 ? 16 - k_ : k_));
        // (2) clusters, smallest first; at equal size the warp-specialised cluster kernel, larger tile first
        if (q.cl > 1) return 200000000LL + q.cl * 1000 + (q.ws ? 100 - k_ : 500 + k_);
        if (q.csm) return ((q.ws && k_ <= 16) ? 100000000LL : 300000000LL) + k_ * 100 + (1 - q.ws);
        return ((long long)(1 - q.ws) * 1000000 + dk * 1000 + k_) * 10 - q.minb;
      };
      const long long score = score_of(t);
      const long long bscore = best < 0 ? 0 : score_of(tiles[best]);
      if (best < 0 || score < bscore) {
        best = i; blay = lo; bl = la; bpack = gsel; bcm = cmsel;
      }
    }
    if (best < 0 && dofs_per_thread > 1)
      return fail(ctx, HZ_EUNSUPPORTED, "hz_partition: no compiled register-blocked kernel with that many DOFs per thread fits this subdomain");
    if (best >= 0 && complex_f)
      return fail(ctx, HZ_EUNSUPPORTED, "hz_partition: complex f is only supported by the one-DOF-per-thread variant");
    if (best < 0 && N > 1024) streamed = true;  // state does not fit on chip: streamed fallback
  }
  if (quad) {
  } else if (best >= 0) {
    ctx->lay = blay; ctx->launch = bl;
    ctx->mx = tiles[best].mx; ctx->my = tiles[best].my; ctx->csm = tiles[best].csm; ctx->ws = tiles[best].ws;
    ctx->cl = tiles[best].cl;
    ctx->pack = tiles[best].pk ? bpack : 1;
    ctx->pk = tiles[best].pk;
    ctx->cmerge = bcm;
    ctx->entry = best;
    // warp-role order of k_sweep_ws: a 3-warp block (2 bulk + 1 edge) puts its edge warp in the middle, so that the bulk
    // warps of the blocks resident on an SM (consecutive hardware warp slots, slot mod 4 = sub-partition) spread evenly
    // over the 4 schedulers (measured: config 2 fp32 0.147 -> 0.111 ms per sweep, config 3 fp32 1.273 -> 1.241 ms)
    ctx->worder = fl.warp_order > 0 ? fl.warp_order - 1 : ((ctx->ws && ctx->cl == 1 && bl.threads == 96) ? 1 : 0);
  } else if (streamed) {
    lay.variant = 2; lay.NT = N < 1024 ? roundup(N, 32) : 1024; lay.NS = roundup(N, 32); lay.TX = lay.TY = 1;
    lay.ntx = lay.nty = 0;
    ctx->lay = lay; ctx->mx = ctx->my = 0; ctx->csm = 0; ctx->ws = 0; ctx->cl = 1;
    ctx->launch.blocks = ctx->L; ctx->launch.threads = lay.NT; ctx->launch.smem = 0;
  } else {
    lay.variant = 0; lay.NT = roundup(N, 32); lay.NS = lay.NT; lay.TX = lay.TY = 1; lay.ntx = lay.nty = 0;
    ctx->lay = lay; ctx->mx = ctx->my = 0; ctx->csm = 0; ctx->ws = 0;
    ctx->launch.blocks = ctx->L; ctx->launch.threads = lay.NT;
    ctx->launch.smem = tab_bytes + 2 * (size_t)(lnx + 2 * P) * (lny + 2 * P) * rs;
  }

  // --- host tables ---
  std::vector<double> tab((size_t)n_t * 4);
  const double tan2 = std::tan(M_PI / n_t) * std::tan(M_PI / n_t);
  for (int nu = 0; nu < n_t; ++nu) {
    tab[4 * nu + 0] = std::cos(2.0 * M_PI * nu / n_t);
    tab[4 * nu + 1] = std::sin(2.0 * M_PI * nu / n_t);
    tab[4 * nu + 2] = std::cos(2.0 * M_PI * nu / n_t) - 0.25 + 0.25 * tan2;                       // kappa_nu
    tab[4 * nu + 3] = (std::cos(2.0 * M_PI * (nu + 0.5) / n_t) - 0.25 + 0.25 * tan2) / ctx->omega;  // kappa_{nu+1/2}/omega
  }
  for (int nu = 0; nu < n_t && nu < kTabCMax; ++nu) {
    ctx->tc32.t[nu] = Tab4<float>{(float)tab[4 * nu], (float)tab[4 * nu + 1], (float)tab[4 * nu + 2], (float)tab[4 * nu + 3]};
    ctx->tc64.t[nu] = Tab4<double>{tab[4 * nu], tab[4 * nu + 1], tab[4 * nu + 2], tab[4 * nu + 3]};
  }
  std::vector<double> bandx, bandy, wxl, wyl;
  make_band(ctx->gll, ctx->ex, ctx->hx, &bandx, &wxl);
  make_band(ctx->gll, ctx->ey, ctx->hy, &bandy, &wyl);
  fill_elem1d<double>(ctx->gll, ctx->hx, &ctx->ex1);
  fill_elem1d<double>(ctx->gll, ctx->hy, &ctx->ey1);

  // --- device allocation ---
  const size_t LS = (size_t)ctx->L * ctx->lay.NS;
  const size_t lam_n = (size_t)ctx->L * 8 * ctx->E, edge_n = (size_t)ctx->L * 4 * ctx->E;
  size_t ws = 0;
  auto alloc0 = [&](void **ptr, size_t bytes) -> cudaError_t {
    cudaError_t e = cudaMalloc(ptr, bytes);
    if (e != cudaSuccess) return e;
    ws += bytes;
    return cudaMemset(*ptr, 0, bytes);
  };
  const bool need_im = ctx->d_fim != nullptr || ctx->d_bc != nullptr;
  HZ_CUDA(alloc0(&ctx->d_gamma, LS * rs));
  HZ_CUDA(alloc0(&ctx->d_alpha, LS * rs));
  HZ_CUDA(alloc0(&ctx->d_bbf_re, LS * rs));
  if (need_im) HZ_CUDA(alloc0(&ctx->d_bbf_im, LS * rs));
  if (ctx->lay.variant == 2) HZ_CUDA(alloc0(&ctx->d_scr, 7 * LS * rs));
  if (ctx->lay.variant == 3) HZ_CUDA(alloc0(&ctx->d_G, (size_t)ctx->L * 3 * (P + 1) * (P + 1) * ctx->launch.threads * rs));
  HZ_CUDA(alloc0(&ctx->d_lam, (lam_n + 2 * LS) * rs));  // joint state: lambda | u_l, one flat array
  ctx->d_usub = (char *)ctx->d_lam + lam_n * rs;
  ctx->n_state = (long long)(lam_n + 2 * LS);
  HZ_CUDA(alloc0(&ctx->d_g, lam_n * rs));
  HZ_CUDA(alloc0(&ctx->d_k2, edge_n * rs));
  HZ_CUDA(alloc0(&ctx->d_bs, edge_n * rs));
  HZ_CUDA(alloc0((void **)&ctx->d_ures, (size_t)2 * ctx->npx * ctx->npy * sizeof(double)));
  if (prec == HZ_F32) {
    HZ_CUDA(upload_as<float>(tab, &ctx->d_tab));
    HZ_CUDA(upload_as<float>(bandx, &ctx->d_bandx));
    HZ_CUDA(upload_as<float>(bandy, &ctx->d_bandy));
  } else {
    HZ_CUDA(upload_as<double>(tab, &ctx->d_tab));
    HZ_CUDA(upload_as<double>(bandx, &ctx->d_bandx));
    HZ_CUDA(upload_as<double>(bandy, &ctx->d_bandy));
  }
  HZ_CUDA(upload_as<double>(wxl, (void **)&ctx->d_wxl));
  HZ_CUDA(upload_as<double>(wyl, (void **)&ctx->d_wyl));
  HZ_CUDA(upload_gather_tables(ctx));
  ctx->ws_bytes = ws;
  ctx->part = true;
  hz_status st = prec == HZ_F32 ? run_build<float>(ctx, 0, 0) : run_build<double>(ctx, 0, 0);
  if (st != HZ_OK) { free_partition(ctx); return st; }
  HZ_CUDA(cudaStreamSynchronize(0));
  if (info_out) {
    hz_part_info inf{};
    inf.n_t = n_t; inf.dofs_per_sub = N; inf.edge_nodes_x = lnx; inf.edge_nodes_y = lny; inf.edge_stride = ctx->E;
    inf.threads_per_block = ctx->launch.threads; inf.blocks = ctx->L;
    inf.dofs_per_thread = ctx->lay.variant == 0 ? 1 : (ctx->lay.variant == 2 ? -1 : ctx->lay.TX * ctx->lay.TY);
    if (ctx->lay.variant == 3) inf.dofs_per_thread = (P + 1) * (P + 1);  // incl. the replicated shared nodes
    inf.tile_mx = ctx->mx; inf.tile_my = ctx->my; inf.cluster_size = ctx->lay.variant == 1 ? ctx->cl : 1;
    inf.subs_per_block = ctx->lay.variant == 1 ? ctx->pack : 1;
    inf.dt = ctx->dt; inf.theta = ctx->theta; inf.sigma = ctx->sigma;
    inf.smem_bytes = ctx->launch.smem; inf.workspace_bytes = ws;
    const char *kn = "k_sweep_dof";
    if (ctx->lay.variant == 3) kn = "k_sweep_quad";
    else if (ctx->lay.variant == 2) kn = "k_sweep_stream";
    else if (ctx->lay.variant == 1)
      kn = ctx->pk ? "k_sweep_pack" : (ctx->cl > 1 ? (ctx->ws ? "k_sweep_cw" : "k_sweep_cl") : (ctx->ws ? "k_sweep_ws" : "k_sweep_tile"));
    std::snprintf(inf.kernel, sizeof(inf.kernel), "%s", kn);
    *info_out = inf;
  }
  return HZ_OK;
}

hz_status hz_ddm_solve(hz_ctx *ctx, const hz_solve_opts *opts, void *u_out, hz_solve_info *info, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!opts) return fail(ctx, HZ_EINVAL, "hz_ddm_solve: NULL opts");
  if (!ctx->part) return fail(ctx, HZ_ESTATE, "hz_ddm_solve: call hz_partition first");
  if (opts->n_outer_max < 0 || opts->n_wh < 1 || !(opts->relax > 0.0) || opts->relax > 1.0)
    return fail(ctx, HZ_EINVAL, "hz_ddm_solve: need n_outer_max >= 0, n_wh >= 1, relax in (0,1]");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t rs = ctx->prec == HZ_F32 ? 4 : 8;
  if (opts->reset_state) {
    HZ_CUDA(cudaMemsetAsync(ctx->d_lam, 0, (size_t)ctx->L * 8 * ctx->E * rs, st));
    HZ_CUDA(cudaMemsetAsync(ctx->d_g, 0, (size_t)ctx->L * 8 * ctx->E * rs, st));
    HZ_CUDA(cudaMemsetAsync(ctx->d_usub, 0, (size_t)2 * ctx->L * ctx->lay.NS * rs, st));
  }
  const int n = opts->n_outer_max;
  const bool checking = opts->tol > 0.0 && opts->check_every > 0;
  const bool graph = opts->use_graph && n > 1;
  // plain launches: three events per sweep (before the sweep, between sweep and exchange, after the exchange), so
  // that the residual checks between two sweeps are not billed to the sweep; [3n] = start of the call
  std::vector<cudaEvent_t> ev(graph ? (size_t)1 : (size_t)3 * n + 1);
  const size_t ev_start = graph ? 0 : (size_t)3 * n;
  for (auto &e : ev) HZ_CUDA(cudaEventCreate(&e));
  auto cleanup = [&]() { for (auto &e : ev) cudaEventDestroy(e); };
  double rel = -1.0;
  int done = 0, other = 0, nexch = 0;
  cudaError_t ce = cudaSuccess;
  hz_status status = HZ_OK;
  auto check = [&]() -> int {  // 1 = converged, 0 = go on, -1 = error (status / ce set)
    ce = launch_gather(ctx, ctx->d_ures, HZ_F64, st);
    if (ce != cudaSuccess) return -1;
    status = residual_impl(ctx, ctx->d_ures, HZ_F64, &rel, st);
    other += 3;
    if (status != HZ_OK) return -1;
    return rel <= opts->tol ? 1 : 0;
  };
  if (graph) {
    int chunk = checking ? opts->check_every : 64;
    if (chunk > n) chunk = n;
    if (!ctx->g_exec || ctx->g_chunk != chunk || ctx->g_nwh != opts->n_wh || ctx->g_warm != opts->warm_start ||
        ctx->g_relax != opts->relax) {
      if (ctx->g_exec) { cudaGraphExecDestroy(ctx->g_exec); ctx->g_exec = nullptr; }
      cudaGraph_t gr = nullptr;
      if (!ctx->cap_stream) ce = cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking);
      if (ce != cudaSuccess) { cleanup(); return cuda_fail(ctx, ce, "hz_ddm_solve (capture stream)"); }
      ce = cudaStreamBeginCapture(ctx->cap_stream, cudaStreamCaptureModeThreadLocal);
      for (int it = 0; it < chunk && ce == cudaSuccess; ++it) {
        ce = launch_sweep(ctx, opts, ctx->cap_stream);
        if (ce == cudaSuccess) ce = launch_exchange(ctx, opts->relax, ctx->cap_stream);
      }
      cudaError_t ce2 = cudaStreamEndCapture(ctx->cap_stream, &gr);
      if (ce == cudaSuccess) ce = ce2;
      if (ce == cudaSuccess) ce = cudaGraphInstantiate(&ctx->g_exec, gr, 0);
      if (gr) cudaGraphDestroy(gr);
      if (ce != cudaSuccess) { cleanup(); return cuda_fail(ctx, ce, "hz_ddm_solve (graph capture)"); }
      ctx->g_chunk = chunk; ctx->g_nwh = opts->n_wh; ctx->g_warm = opts->warm_start; ctx->g_relax = opts->relax;
    }
    ce = cudaEventRecord(ev[ev_start], st);
    while (done < n && ce == cudaSuccess) {
      const int m = n - done < chunk ? n - done : chunk;
      if (m == chunk) {
        ce = cudaGraphLaunch(ctx->g_exec, st);
      } else {
        for (int it = 0; it < m && ce == cudaSuccess; ++it) {
          ce = launch_sweep(ctx, opts, st);
          if (ce == cudaSuccess) ce = launch_exchange(ctx, opts->relax, st);
        }
      }
      if (ce != cudaSuccess) break;
      done += m; nexch += m;
      if (checking) {
        const int c = check();
        if (c < 0) { if (status != HZ_OK) { cleanup(); return status; } break; }
        if (c > 0) break;
      }
    }
  } else {
    ce = cudaEventRecord(ev[ev_start], st);
    for (int it = 0; it < n && ce == cudaSuccess; ++it) {
      ce = cudaEventRecord(ev[3 * it], st);
      if (ce != cudaSuccess) break;
      ce = launch_sweep(ctx, opts, st);
      if (ce != cudaSuccess) break;
      ce = cudaEventRecord(ev[3 * it + 1], st);
      if (ce != cudaSuccess) break;
      ce = launch_exchange(ctx, opts->relax, st);
      if (ce != cudaSuccess) break;
      ++nexch;
      ce = cudaEventRecord(ev[3 * it + 2], st);
      if (ce != cudaSuccess) break;
      ++done;
      if (checking && (done % opts->check_every == 0 || done == n)) {
        const int c = check();
        if (c < 0) { if (status != HZ_OK) { cleanup(); return status; } break; }
        if (c > 0) break;
      }
    }
  }
  if (ce == cudaSuccess && u_out) { ce = launch_gather(ctx, u_out, ctx->prec, st); ++other; }
  cudaEvent_t ev_end;
  if (ce == cudaSuccess) ce = cudaEventCreate(&ev_end);
  if (ce == cudaSuccess) ce = cudaEventRecord(ev_end, st);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
  if (ce != cudaSuccess) { cleanup(); return cuda_fail(ctx, ce, "hz_ddm_solve"); }
  if (info) {
    hz_solve_info inf{};
    inf.n_outer_done = done; inf.n_t = ctx->n_t; inf.rel_residual = rel;
    float ms = 0.f;
    if (graph) {
      inf.sweep_ms_total = -1.0;
      inf.exch_ms_total = -1.0;
    } else {
      for (int it = 0; it < done; ++it) {
        cudaEventElapsedTime(&ms, ev[3 * it], ev[3 * it + 1]);
        inf.sweep_ms_total += ms;
        cudaEventElapsedTime(&ms, ev[3 * it + 1], ev[3 * it + 2]);
        inf.exch_ms_total += ms;
      }
    }
    cudaEventElapsedTime(&ms, ev[ev_start], ev_end);
    inf.total_ms = ms;
    inf.dof_timesteps = (double)ctx->L * ctx->lay.lnx * ctx->lay.lny * (double)opts->n_wh * (ctx->n_t - 1) * done;
    inf.sweep_launches = done; inf.exch_launches = nexch; inf.other_launches = other;
    *info = inf;
  }
  cudaEventDestroy(ev_end);
  cleanup();
  return HZ_OK;
}

hz_status hz_operator_time(hz_ctx *ctx, const void *u_dev, hz_prec prec, int reps, void *y_dev, double *ms_per_eval,
                           void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!u_dev || !ms_per_eval || reps < 1) return fail(ctx, HZ_EINVAL, "hz_operator_time: NULL argument or reps < 1");
  if (prec != HZ_F32 && prec != HZ_F64) return fail(ctx, HZ_EINVAL, "hz_operator_time: bad precision");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t nn = (size_t)ctx->npx * ctx->npy, rs = prec == HZ_F32 ? 4 : 8;
  EventGuard e0, e1;
  HZ_CUDA(cudaEventCreate(&e0.e));
  HZ_CUDA(cudaEventCreate(&e1.e));
  if (ctx->general) {  // general quads: the fp64 residual kernel is the operator kernel (no separate output pass)
    if (prec != HZ_F64 || y_dev) return fail(ctx, HZ_EUNSUPPORTED, "hz_operator_time: general quadrilaterals: HZ_F64 only, no output vector");
    double rel = 0.0;
    hz_status s0 = residual_impl(ctx, u_dev, HZ_F64, &rel, st);  // allocates the partial-sum buffers, warm-up
    if (s0 != HZ_OK) return s0;
    const int bs = 256, nb = (int)((nn + bs - 1) / bs);
    const Geo g = make_geo(ctx);
    HZ_CUDA(cudaEventRecord(e0.e, st));
    for (int r = 0; r < reps; ++r)
      k_residual_quad<double><<<nb, bs, 0, st>>>(g, ctx->refq, ctx->d_vx, ctx->d_vy, ctx->d_c, ctx->d_fre, ctx->d_fim, ctx->d_bc,
                                                 (const double *)u_dev, ctx->d_part);
  } else {
    // w^2 / c^2 in the operator's precision and the output vector y, owned by the context
    if (!ctx->d_opk2 || ctx->op_prec != (int)prec) {
      if (ctx->d_opk2) cudaFree(ctx->d_opk2);
      if (ctx->d_opy) cudaFree(ctx->d_opy);
      ctx->d_opk2 = ctx->d_opy = nullptr;
      HZ_CUDA(cudaMalloc(&ctx->d_opk2, nn * rs));
      HZ_CUDA(cudaMalloc(&ctx->d_opy, 2 * nn * rs));
      ctx->op_prec = (int)prec;
      const unsigned nbk = (unsigned)((nn + 255) / 256);
      if (prec == HZ_F32) k_helm_k2<float><<<nbk, 256, 0, st>>>((long long)nn, ctx->omega, ctx->d_c, (float *)ctx->d_opk2);
      else k_helm_k2<double><<<nbk, 256, 0, st>>>((long long)nn, ctx->omega, ctx->d_c, (double *)ctx->d_opk2);
      HZ_CUDA(cudaGetLastError());
    }
    void *yv = y_dev ? y_dev : ctx->d_opy;
    auto once = [&]() -> cudaError_t {
      if (prec == HZ_F32) return launch_helm<float, float, 1>(ctx, (const float *)ctx->d_opk2, u_dev, nullptr, (float *)yv, st);
      return launch_helm<double, double, 1>(ctx, (const double *)ctx->d_opk2, u_dev, nullptr, (double *)yv, st);
    };
    HZ_CUDA(once());  // warm-up
    HZ_CUDA(cudaEventRecord(e0.e, st));
    for (int r = 0; r < reps; ++r) HZ_CUDA(once());
  }
  HZ_CUDA(cudaEventRecord(e1.e, st));
  HZ_CUDA(cudaStreamSynchronize(st));
  float ms = 0.f;
  HZ_CUDA(cudaEventElapsedTime(&ms, e0.e, e1.e));
  *ms_per_eval = ms / reps;
  return HZ_OK;
}

hz_status hz_ddm_solve_sources(hz_ctx *ctx, const hz_solve_opts *opts, int n_src, const double *const *f_re_host,
                               void *const *u_host, hz_sources_info *info, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!opts || !f_re_host || !u_host || n_src < 1) return fail(ctx, HZ_EINVAL, "hz_ddm_solve_sources: NULL argument or n_src < 1");
  if (!ctx->part) return fail(ctx, HZ_ESTATE, "hz_ddm_solve_sources: call hz_partition first");
  if (opts->n_outer_max < 1 || opts->n_wh < 1 || !(opts->relax > 0.0) || opts->relax > 1.0)
    return fail(ctx, HZ_EINVAL, "hz_ddm_solve_sources: need n_outer_max >= 1, n_wh >= 1, relax in (0,1]");
  if (ctx->d_fim) return fail(ctx, HZ_EUNSUPPORTED, "hz_ddm_solve_sources: real sources only (the context has an imaginary part)");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t rs = ctx->prec == HZ_F32 ? 4 : 8;
  const size_t nn = (size_t)ctx->npx * ctx->npy;
  if (!ctx->s_in) {
    HZ_CUDA(cudaStreamCreateWithFlags(&ctx->s_in, cudaStreamNonBlocking));
    HZ_CUDA(cudaStreamCreateWithFlags(&ctx->s_out, cudaStreamNonBlocking));
    for (int b = 0; b < 2; ++b) {
      HZ_CUDA(cudaMalloc((void **)&ctx->d_fstage[b], nn * sizeof(double)));
      HZ_CUDA(cudaEventCreateWithFlags(&ctx->ev_up[b], cudaEventDisableTiming));
      HZ_CUDA(cudaEventCreateWithFlags(&ctx->ev_build[b], cudaEventDisableTiming));
      HZ_CUDA(cudaEventCreateWithFlags(&ctx->ev_gather[b], cudaEventDisableTiming));
      HZ_CUDA(cudaEventCreateWithFlags(&ctx->ev_down[b], cudaEventDisableTiming));
    }
  }
  if (ctx->ubuf_bytes != 2 * nn * rs) {  // the gathered field has the partition's precision, which may have changed
    for (int b = 0; b < 2; ++b) {
      if (ctx->d_ubuf[b]) cudaFree(ctx->d_ubuf[b]);
      ctx->d_ubuf[b] = nullptr;
      HZ_CUDA(cudaMalloc(&ctx->d_ubuf[b], 2 * nn * rs));
    }
    ctx->ubuf_bytes = 2 * nn * rs;
  }
  cudaEvent_t e0, e1;
  HZ_CUDA(cudaEventCreate(&e0));
  HZ_CUDA(cudaEventCreate(&e1));
  cudaError_t ce = cudaEventRecord(e0, st);
  if (ce == cudaSuccess) ce = cudaStreamWaitEvent(ctx->s_in, e0, 0);
  int launches = 0;
  for (int s = 0; s < n_src && ce == cudaSuccess; ++s) {
    const int b = s & 1;
    if (!f_re_host[s] || !u_host[s]) { ce = cudaErrorInvalidValue; break; }
    // copy-in stream: source s into staging buffer b, once the build of source s-2 has consumed it
    if (s >= 2) ce = cudaStreamWaitEvent(ctx->s_in, ctx->ev_build[b], 0);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(ctx->d_fstage[b], f_re_host[s], nn * sizeof(double), cudaMemcpyHostToDevice, ctx->s_in);
    if (ce == cudaSuccess) ce = cudaEventRecord(ctx->ev_up[b], ctx->s_in);
    // compute stream: rebuild beta*b from the staged source, sweeps, gather
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(st, ctx->ev_up[b], 0);
    if (ce != cudaSuccess) break;
    hz_status bst = ctx->prec == HZ_F32 ? run_build<float>(ctx, 1, st, ctx->d_fstage[b]) : run_build<double>(ctx, 1, st, ctx->d_fstage[b]);
    if (bst != HZ_OK) {
      cudaStreamSynchronize(ctx->s_in); cudaStreamSynchronize(ctx->s_out); cudaStreamSynchronize(st);
      cudaEventDestroy(e0); cudaEventDestroy(e1);
      return bst;
    }
    ce = cudaEventRecord(ctx->ev_build[b], st);
    ++launches;
    if (ce == cudaSuccess && opts->reset_state) {
      ce = cudaMemsetAsync(ctx->d_lam, 0, (size_t)ctx->n_state * rs, st);
      if (ce == cudaSuccess) ce = cudaMemsetAsync(ctx->d_g, 0, (size_t)ctx->L * 8 * ctx->E * rs, st);
    }
    for (int it = 0; it < opts->n_outer_max && ce == cudaSuccess; ++it) {
      ce = launch_sweep(ctx, opts, st);
      if (ce == cudaSuccess) ce = launch_exchange(ctx, opts->relax, st);
      launches += 2;
    }
    if (ce == cudaSuccess && s >= 2) ce = cudaStreamWaitEvent(st, ctx->ev_down[b], 0);  // field buffer b is free again
    if (ce == cudaSuccess) ce = launch_gather(ctx, ctx->d_ubuf[b], ctx->prec, st);
    ++launches;
    if (ce == cudaSuccess) ce = cudaEventRecord(ctx->ev_gather[b], st);
    // copy-out stream: field s to the host
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(ctx->s_out, ctx->ev_gather[b], 0);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(u_host[s], ctx->d_ubuf[b], 2 * nn * rs, cudaMemcpyDeviceToHost, ctx->s_out);
    if (ce == cudaSuccess) ce = cudaEventRecord(ctx->ev_down[b], ctx->s_out);
  }
  // the context keeps the last source (hz_residual and later hz_ddm_solve calls see it)
  if (ce == cudaSuccess) ce = cudaMemcpyAsync(ctx->d_fre, ctx->d_fstage[(n_src - 1) & 1], nn * sizeof(double), cudaMemcpyDeviceToDevice, st);
  if (ce == cudaSuccess) ce = cudaStreamWaitEvent(st, ctx->ev_down[(n_src - 1) & 1], 0);
  if (ce == cudaSuccess && n_src >= 2) ce = cudaStreamWaitEvent(st, ctx->ev_down[n_src & 1], 0);
  if (ce == cudaSuccess) ce = cudaEventRecord(e1, st);
  if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
  float ms = 0.f;
  if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (ce != cudaSuccess) {
    cudaStreamSynchronize(ctx->s_in); cudaStreamSynchronize(ctx->s_out); cudaStreamSynchronize(st);
    return cuda_fail(ctx, ce, "hz_ddm_solve_sources");
  }
  if (info) {
    info->sources_done = n_src;
    info->total_ms = ms;
    info->dof_timesteps = (double)ctx->L * ctx->lay.lnx * ctx->lay.lny * (double)opts->n_wh * (ctx->n_t - 1) * opts->n_outer_max * n_src;
    info->launches = launches;
    info->h2d_bytes = (double)n_src * nn * sizeof(double);
    info->d2h_bytes = (double)n_src * 2 * nn * rs;
  }
  return HZ_OK;
}

}  // extern "C"

namespace {

template <typename real>
hz_status gmres_impl(hz_ctx *ctx, const hz_gmres_opts *o, void *u_out, hz_gmres_info *info, cudaStream_t st) {
  // lambda_only: the vectors are the lambda part of the joint state (the first L*8*E reals of d_lam), sweeps cold-started
  const bool lam_only = o->lambda_only != 0;
  const long long n = lam_only ? (long long)ctx->L * 8 * ctx->E : ctx->n_state;
  const int m = o->restart;
  const int nvec = m + 3;  // V_0..V_m, c, x
  const size_t rs = sizeof(real);
  const int bs = 256, nblk = 592;  // 4 blocks per SM on 148 SMs
  if (!ctx->d_kry || ctx->kry_vecs < nvec || ctx->kry_len < n) {
    if (ctx->d_kry) cudaFree(ctx->d_kry);
    if (ctx->d_kpart) cudaFree(ctx->d_kpart);
    ctx->d_kry = nullptr; ctx->d_kpart = nullptr; ctx->kry_vecs = 0;
    HZ_CUDA(cudaMalloc(&ctx->d_kry, (size_t)nvec * n * rs));
    HZ_CUDA(cudaMalloc((void **)&ctx->d_kpart, ((size_t)(m + 2) * nblk + 2 * (m + 2)) * sizeof(double)));
    ctx->kry_vecs = nvec;
    ctx->kry_len = n;
  }
  real *V = (real *)ctx->d_kry, *cvec = V + (size_t)(m + 1) * n, *x = cvec + n, *state = (real *)ctx->d_lam;
  double *part = ctx->d_kpart, *dres = part + (size_t)(m + 2) * nblk, *dcoef = dres + (m + 2);
  hz_solve_opts so{};
  so.n_wh = o->n_wh; so.warm_start = lam_only ? 0 : 1; so.relax = o->relax;
  int sweeps = 0;
  auto sweep = [&]() -> cudaError_t {
    cudaError_t e = launch_sweep(ctx, &so, st);
    if (e == cudaSuccess) e = launch_exchange(ctx, o->relax, st);
    ++sweeps;
    return e;
  };
  // lambda_only: u_l of the lambda now in the state -- the sweep kernel without the exchange (lambda is not advanced),
  // then n_polish warm-started WaveHoltz iterations at that lambda
  auto materialise = [&]() -> cudaError_t {
    if (!lam_only) return cudaSuccess;
    cudaError_t e = launch_sweep(ctx, &so, st);
    ++sweeps;
    if (e == cudaSuccess && o->n_polish > 0) {
      hz_solve_opts sp = so;
      sp.n_wh = o->n_polish; sp.warm_start = 1;
      e = launch_sweep(ctx, &sp, st);
      ++sweeps;
    }
    return e;
  };
  std::vector<double> hbuf(m + 2);
  // h[0..nv) = V_i . w  (i < nv), synchronous
  auto dots = [&](const real *Vb, int nv, const real *w, double *h) -> cudaError_t {
    k_dots<real><<<dim3(nblk, nv), bs, 0, st>>>(n, Vb, n, w, part);
    k_reduce_rows<<<nv, 256, 0, st>>>(part, nblk, dres);
    cudaError_t e = cudaMemcpyAsync(h, dres, nv * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e;
  };
  auto axpys = [&](real *w, const real *Vb, int nv, const double *coef) -> cudaError_t {
    cudaError_t e = cudaMemcpyAsync(dcoef, coef, nv * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    k_axpys<real><<<nblk, bs, 0, st>>>(n, w, Vb, n, nv, dcoef);
    return cudaGetLastError();
  };
  EventGuard e0, e1;  // destroyed on every return path
  HZ_CUDA(cudaEventCreate(&e0.e));
  HZ_CUDA(cudaEventCreate(&e1.e));
  HZ_CUDA(cudaEventRecord(e0.e, st));
  // x0 and c = F(0)
  if (o->reset_state) HZ_CUDA(cudaMemsetAsync(x, 0, n * rs, st));
  else HZ_CUDA(cudaMemcpyAsync(x, state, n * rs, cudaMemcpyDeviceToDevice, st));
  HZ_CUDA(cudaMemsetAsync(state, 0, n * rs, st));
  HZ_CUDA(cudaMemsetAsync(ctx->d_g, 0, (size_t)ctx->L * 8 * ctx->E * rs, st));
  HZ_CUDA(sweep());
  HZ_CUDA(cudaMemcpyAsync(cvec, state, n * rs, cudaMemcpyDeviceToDevice, st));
  double cc = 0.0;
  HZ_CUDA(dots(cvec, 1, cvec, &cc));
  const double cnorm = std::sqrt(cc);
  int steps = 0, cycles = 0;
  double lin = 1.0, rel = -1.0;
  bool x_is_zero = o->reset_state != 0;
  std::vector<double> H((size_t)(m + 1) * m), cs(m), sn(m), g(m + 1), y(m), h2(m + 2);
  bool finished = cnorm == 0.0;
  // linear-residual target that ends a cycle when a Helmholtz tolerance is given; tightened whenever the true
  // residual (checked at the end of the cycle) turns out to be above the tolerance
  double lin_target = 0.5 * o->tol;
  while (!finished && steps < o->max_steps) {
    // r = F(x) - x  (= c for x = 0)
    if (x_is_zero) {
      HZ_CUDA(cudaMemcpyAsync(V, cvec, n * rs, cudaMemcpyDeviceToDevice, st));
    } else {
      HZ_CUDA(cudaMemcpyAsync(state, x, n * rs, cudaMemcpyDeviceToDevice, st));
      HZ_CUDA(sweep());
      k_lincomb<real><<<nblk, bs, 0, st>>>(n, V, 1.0, state, -1.0, x, 0.0, nullptr);
      HZ_CUDA(cudaGetLastError());
    }
    double bb = 0.0;
    HZ_CUDA(dots(V, 1, V, &bb));
    const double beta = std::sqrt(bb);
    if (beta == 0.0) break;
    k_lincomb<real><<<nblk, bs, 0, st>>>(n, V, 1.0 / beta, V, 0.0, V, 0.0, nullptr);
    HZ_CUDA(cudaGetLastError());
    std::fill(g.begin(), g.end(), 0.0);
    g[0] = beta;
    const int mc = m < o->max_steps - steps ? m : o->max_steps - steps;
    int k = 0;
    for (int j = 0; j < mc; ++j) {
      real *vj = V + (size_t)j * n, *w = V + (size_t)(j + 1) * n;
      // w = (I - T) v_j = v_j - (F(v_j) - c)
      HZ_CUDA(cudaMemcpyAsync(state, vj, n * rs, cudaMemcpyDeviceToDevice, st));
      HZ_CUDA(sweep());
      k_lincomb<real><<<nblk, bs, 0, st>>>(n, w, 1.0, vj, -1.0, state, 1.0, cvec);
      HZ_CUDA(cudaGetLastError());
      // classical Gram-Schmidt, twice
      double *hc = &H[(size_t)j * (m + 1)];  // column j, rows 0..j+1
      HZ_CUDA(dots(V, j + 1, w, hbuf.data()));
      for (int i = 0; i <= j; ++i) { hc[i] = hbuf[i]; h2[i] = -hbuf[i]; }
      HZ_CUDA(axpys(w, V, j + 1, h2.data()));
      HZ_CUDA(dots(V, j + 1, w, hbuf.data()));
      for (int i = 0; i <= j; ++i) { hc[i] += hbuf[i]; h2[i] = -hbuf[i]; }
      HZ_CUDA(axpys(w, V, j + 1, h2.data()));
      double ww = 0.0;
      HZ_CUDA(dots(w, 1, w, &ww));
      hc[j + 1] = std::sqrt(ww);
      if (hc[j + 1] > 0.0) {
        k_lincomb<real><<<nblk, bs, 0, st>>>(n, w, 1.0 / hc[j + 1], w, 0.0, w, 0.0, nullptr);
        HZ_CUDA(cudaGetLastError());
      }
      for (int i = 0; i < j; ++i) {  // previous Givens rotations on the new column
        const double t = cs[i] * hc[i] + sn[i] * hc[i + 1];
        hc[i + 1] = -sn[i] * hc[i] + cs[i] * hc[i + 1];
        hc[i] = t;
      }
      const double d = std::hypot(hc[j], hc[j + 1]);
      cs[j] = hc[j] / d; sn[j] = hc[j + 1] / d;
      hc[j] = d; hc[j + 1] = 0.0;
      g[j + 1] = -sn[j] * g[j];
      g[j] = cs[j] * g[j];
      k = j + 1;
      ++steps;
      lin = std::fabs(g[j + 1]) / cnorm;
      if (o->lin_history && steps <= o->history_len) o->lin_history[steps - 1] = lin;
      if ((o->lin_tol > 0.0 && lin <= o->lin_tol) || (o->tol > 0.0 && lin <= lin_target)) break;
    }
    // y = R^-1 g (back substitution), x += V y
    for (int i = k - 1; i >= 0; --i) {
      double sacc = g[i];
      for (int q = i + 1; q < k; ++q) sacc -= H[(size_t)q * (m + 1) + i] * y[q];
      y[i] = sacc / H[(size_t)i * (m + 1) + i];
    }
    HZ_CUDA(axpys(x, V, k, y.data()));
    x_is_zero = false;
    ++cycles;
    if (o->lin_tol > 0.0 && lin <= o->lin_tol) finished = true;
    if (o->tol > 0.0 && lin <= lin_target) {
      HZ_CUDA(cudaMemcpyAsync(state, x, n * rs, cudaMemcpyDeviceToDevice, st));
      HZ_CUDA(materialise());
      HZ_CUDA(launch_gather(ctx, ctx->d_ures, HZ_F64, st));
      hz_status s2 = residual_impl(ctx, ctx->d_ures, HZ_F64, &rel, st);
      if (s2 != HZ_OK) return s2;
      if (rel <= o->tol) finished = true;
      else lin_target *= std::fmin(0.5, 0.5 * o->tol / rel);
    }
  }
  // leave the iterate in the context's state, report its Helmholtz residual
  HZ_CUDA(cudaMemcpyAsync(state, x, n * rs, cudaMemcpyDeviceToDevice, st));
  HZ_CUDA(materialise());
  HZ_CUDA(launch_gather(ctx, ctx->d_ures, HZ_F64, st));
  {
    hz_status s2 = residual_impl(ctx, ctx->d_ures, HZ_F64, &rel, st);
    if (s2 != HZ_OK) return s2;
  }
  if (u_out) HZ_CUDA(launch_gather(ctx, u_out, ctx->prec, st));
  HZ_CUDA(cudaEventRecord(e1.e, st));
  HZ_CUDA(cudaStreamSynchronize(st));
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0.e, e1.e);
  if (info) {
    hz_gmres_info inf{};
    inf.steps_done = steps; inf.sweeps_done = sweeps; inf.cycles = cycles; inf.lin_residual = lin;
    inf.rel_residual = rel; inf.total_ms = ms; inf.krylov_bytes = (size_t)nvec * n * rs;
    *info = inf;
  }
  return HZ_OK;
}

}  // namespace

namespace {

inline cudaError_t launch_minres(const MinresArgs<float> &a, int p, SweepLaunch c, cudaStream_t st) { return launch_minres_f32(a, p, c, st); }
inline cudaError_t launch_minres(const MinresArgs<double> &a, int p, SweepLaunch c, cudaStream_t st) { return launch_minres_f64(a, p, c, st); }
inline cudaError_t launch_minres_tile(const MinresArgs<float> &a, const Elem1D<float> &x, const Elem1D<float> &y, int p, int m,
                                      SweepLaunch c, cudaStream_t st) { return launch_minres_tile_f32(a, x, y, p, m, c, st); }
inline cudaError_t launch_minres_tile(const MinresArgs<double> &a, const Elem1D<double> &x, const Elem1D<double> &y, int p, int m,
                                      SweepLaunch c, cudaStream_t st) { return launch_minres_tile_f64(a, x, y, p, m, c, st); }

template <typename real>
hz_status minres_impl(hz_ctx *ctx, const hz_minres_opts *o, int *iters_out, double *res_out, hz_minres_info *info,
                      cudaStream_t st) {
  const size_t LS = (size_t)ctx->L * ctx->lay.NS, EN = (size_t)ctx->L * 4 * ctx->E;
  if (!ctx->d_mr) {
    HZ_CUDA(cudaMalloc(&ctx->d_mr, (5 * LS + EN) * sizeof(real)));
    HZ_CUDA(cudaMemset(ctx->d_mr, 0, (5 * LS + EN) * sizeof(real)));
    HZ_CUDA(cudaMalloc((void **)&ctx->d_mr_iters, ctx->L * sizeof(int)));
    HZ_CUDA(cudaMalloc((void **)&ctx->d_mr_res, ctx->L * sizeof(double)));
  }
  real *base = (real *)ctx->d_mr;
  real *mloc = base, *w2M = base + LS, *wH = base + 2 * LS, *bfr = base + 3 * LS, *bfi = base + 4 * LS, *sedge = base + 5 * LS;
  {  // (re)build: the source may have changed through hz_set_source
    const long long total = (long long)ctx->L * ctx->lay.lnx * ctx->lay.lny;
    k_build_minres<real><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(make_geo(ctx), ctx->lay, ctx->d_c, ctx->d_fre,
                                                                         ctx->d_fim, ctx->d_bc, ctx->d_wxl, ctx->d_wyl,
                                                                         mloc, w2M, wH, bfr, bfi, sedge);
    HZ_CUDA(cudaGetLastError());
  }
  MinresArgs<real> a{};
  a.lay = ctx->lay; a.sx = ctx->sx; a.sy = ctx->sy; a.E = ctx->E;
  a.warm = o->warm_start; a.max_iters = o->max_iters; a.tol = (real)o->tol;
  a.mloc = mloc; a.w2M = w2M; a.wH = wH; a.bf_re = bfr;
  a.bf_im = (ctx->d_fim || ctx->d_bc) ? bfi : nullptr;
  a.sedge = sedge;
  a.bandx = (const real *)ctx->d_bandx; a.bandy = (const real *)ctx->d_bandy;
  a.u_sub = (real *)ctx->d_usub; a.lam = (const real *)ctx->d_lam; a.gout = (real *)ctx->d_g;
  a.k2edge = (const real *)ctx->d_k2;
  a.iters = ctx->d_mr_iters; a.res = ctx->d_mr_res;
  SweepLaunch cfg = ctx->launch;
  const int P = ctx->p;
  const bool tiled = ctx->lay.variant == 1;
  Elem1D<real> ex1{}, ey1{};
  if (tiled) {   // the register-blocked layout of the WaveHoltz kernels: one thread per tile, one subdomain per block
    const int v16 = 16 / (int)sizeof(real), T = ctx->lay.TX;
    const int rsw = 4 * ((T + v16 - 1) / v16 * v16) + v16;
    cfg.blocks = ctx->L;
    cfg.threads = roundup(ctx->lay.ntx * ctx->lay.nty, 32);
    cfg.smem = 72 * sizeof(double) + 2 * (size_t)(cfg.threads + 2) * rsw * sizeof(real);
    for (int i = 0; i <= kMaxP; ++i) {
      for (int j = 0; j <= kMaxP; ++j) { ex1.kin[i][j] = (real)ctx->ex1.kin[i][j]; ey1.kin[i][j] = (real)ctx->ey1.kin[i][j]; }
      ex1.k0[i] = (real)ctx->ex1.k0[i]; ex1.kp[i] = (real)ctx->ex1.kp[i];
      ey1.k0[i] = (real)ctx->ey1.k0[i]; ey1.kp[i] = (real)ctx->ey1.kp[i];
    }
  } else {
    cfg.smem = 72 * sizeof(double) + 2 * (size_t)(ctx->lay.lnx + 2 * P) * (ctx->lay.lny + 2 * P) * sizeof(real);
  }
  cudaEvent_t e0, e1;
  HZ_CUDA(cudaEventCreate(&e0));
  HZ_CUDA(cudaEventCreate(&e1));
  HZ_CUDA(cudaEventRecord(e0, st));
  if (tiled) HZ_CUDA(launch_minres_tile(a, ex1, ey1, P, ctx->mx, cfg, st));
  else HZ_CUDA(launch_minres(a, P, cfg, st));
  HZ_CUDA(cudaEventRecord(e1, st));
  if (o->relax > 0.0) HZ_CUDA(launch_exchange(ctx, o->relax, st));
  std::vector<int> hi(ctx->L);
  std::vector<double> hr(ctx->L);
  HZ_CUDA(cudaMemcpyAsync(hi.data(), ctx->d_mr_iters, ctx->L * sizeof(int), cudaMemcpyDeviceToHost, st));
  HZ_CUDA(cudaMemcpyAsync(hr.data(), ctx->d_mr_res, ctx->L * sizeof(double), cudaMemcpyDeviceToHost, st));
  HZ_CUDA(cudaStreamSynchronize(st));
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (iters_out) std::memcpy(iters_out, hi.data(), ctx->L * sizeof(int));
  if (res_out) std::memcpy(res_out, hr.data(), ctx->L * sizeof(double));
  if (info) {
    hz_minres_info inf{};
    double sum = 0.0;
    for (int l = 0; l < ctx->L; ++l) {
      if (hi[l] > inf.iters_max) inf.iters_max = hi[l];
      sum += hi[l];
      if (hr[l] > inf.res_max) inf.res_max = hr[l];
    }
    inf.iters_mean = sum / ctx->L;
    inf.kernel_ms = ms;
    *info = inf;
  }
  return HZ_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------------
// hz_ddm_solve_mixed: defect correction in the DDM state space, X in fp64 on `hi`, corrections in fp32 on `lo`
// (reading R27; oracle: ddm_mixed_cycle)
// ---------------------------------------------------------------------------------------------------------------
extern "C" hz_status hz_ddm_solve_mixed(hz_ctx *lo, hz_ctx *hi, const hz_mixed_opts *opts, double *u_out,
                                        hz_mixed_info *info, void *stream) {
  if (!lo || !hi) return HZ_EINVAL;
  hz_ctx *ctx = hi;  // error messages and the HZ_CUDA macro report on `hi`
  if (!opts) return fail(ctx, HZ_EINVAL, "hz_ddm_solve_mixed: NULL opts");
  if (!lo->part || !hi->part) return fail(ctx, HZ_ESTATE, "hz_ddm_solve_mixed: call hz_partition on both contexts first");
  if (lo->prec != HZ_F32 || hi->prec != HZ_F64)
    return fail(ctx, HZ_ESTATE, "hz_ddm_solve_mixed: `lo` must be partitioned with HZ_F32 and `hi` with HZ_F64");
  if (lo->general || hi->general || lo->d_fim || hi->d_fim)
    return fail(ctx, HZ_EUNSUPPORTED, "hz_ddm_solve_mixed: uniform-mesh contexts with a real source only");
  if (lo->nx != hi->nx || lo->ny != hi->ny || lo->p != hi->p || lo->sx != hi->sx || lo->sy != hi->sy || lo->n_t != hi->n_t ||
      lo->x0 != hi->x0 || lo->x1 != hi->x1 || lo->y0 != hi->y0 || lo->y1 != hi->y1 || lo->omega != hi->omega)
    return fail(ctx, HZ_EINVAL, "hz_ddm_solve_mixed: the two contexts differ in mesh, frequency, partition or N_t");
  if (opts->n_cycles_max < 0 || opts->m_inner < 1 || opts->n_wh < 1 || !(opts->relax > 0.0) || opts->relax > 1.0)
    return fail(ctx, HZ_EINVAL, "hz_ddm_solve_mixed: need n_cycles_max >= 0, m_inner >= 1, n_wh >= 1, relax in (0,1]");
  cudaStream_t st = (cudaStream_t)stream;
  const long long nlam = (long long)hi->L * 8 * hi->E;
  const long long ncan = nlam + (long long)hi->L * 2 * hi->lay.lnx * hi->lay.lny;  // canonical elements of the state
  if (!hi->d_mix) HZ_CUDA(cudaMalloc(&hi->d_mix, (size_t)hi->n_state * sizeof(double)));
  if (!lo->d_mix) {
    HZ_CUDA(cudaMalloc(&lo->d_mix, (size_t)lo->n_state * sizeof(float)));
    HZ_CUDA(cudaMemsetAsync(lo->d_mix, 0, (size_t)lo->n_state * sizeof(float), st));  // padding slots stay zero
  }
  if (!lo->d_bbf_zero) {
    HZ_CUDA(cudaMalloc(&lo->d_bbf_zero, (size_t)lo->L * lo->lay.NS * sizeof(float)));
    HZ_CUDA(cudaMemsetAsync(lo->d_bbf_zero, 0, (size_t)lo->L * lo->lay.NS * sizeof(float), st));
  }
  double *Xold = (double *)hi->d_mix, *Sh = (double *)hi->d_lam;
  float *Dl = (float *)lo->d_mix, *Sl = (float *)lo->d_lam;
  if (opts->reset_state) {
    HZ_CUDA(cudaMemsetAsync(hi->d_lam, 0, (size_t)hi->n_state * sizeof(double), st));
    HZ_CUDA(cudaMemsetAsync(hi->d_g, 0, (size_t)nlam * sizeof(double), st));
  }
  HZ_CUDA(cudaMemsetAsync(lo->d_lam, 0, (size_t)lo->n_state * sizeof(float), st));
  hz_solve_opts so{};
  so.n_wh = opts->n_wh; so.warm_start = 1; so.relax = opts->relax;
  EventGuard e0, e1;
  HZ_CUDA(cudaEventCreate(&e0.e));
  HZ_CUDA(cudaEventCreate(&e1.e));
  HZ_CUDA(cudaEventRecord(e0.e, st));
  const bool checking = opts->tol > 0.0 && opts->check_every > 0;
  const unsigned nbc = (unsigned)((ncan + 255) / 256);
  int cycles = 0, nlo = 0, nhi = 0;
  double rel = -1.0;
  for (int cy = 0; cy < opts->n_cycles_max; ++cy) {
    if (opts->m_inner > 1) HZ_CUDA(cudaMemcpyAsync(Xold, Sh, (size_t)hi->n_state * sizeof(double), cudaMemcpyDeviceToDevice, st));
    HZ_CUDA(launch_sweep(hi, &so, st));                // F(X) at full precision
    HZ_CUDA(launch_exchange(hi, opts->relax, st));
    ++nhi;
    if (opts->m_inner > 1) {
      k_mixed_defect<<<nbc, 256, 0, st>>>(ncan, nlam, hi->lay, lo->lay, Sh, Xold, Sl, Dl);
      HZ_CUDA(cudaGetLastError());
      for (int k = 1; k < opts->m_inner; ++k) {        // delta_{k+1} = T delta_k + D
        HZ_CUDA(launch_sweep(lo, &so, st, /*homog=*/true));
        HZ_CUDA(launch_exchange(lo, opts->relax, st));
        k_add_f32<<<1184, 256, 0, st>>>(lo->n_state, Sl, Dl);
        HZ_CUDA(cudaGetLastError());
        ++nlo;
      }
      k_mixed_update<<<nbc, 256, 0, st>>>(ncan, nlam, hi->lay, lo->lay, Sh, Xold, Sl);
      HZ_CUDA(cudaGetLastError());
    }
    ++cycles;
    if (checking && (cycles % opts->check_every == 0 || cycles == opts->n_cycles_max)) {
      HZ_CUDA(launch_gather(hi, hi->d_ures, HZ_F64, st));
      hz_status s2 = residual_impl(hi, hi->d_ures, HZ_F64, &rel, st);
      if (s2 != HZ_OK) return s2;
      if (rel <= opts->tol) break;
    }
  }
  if (u_out) HZ_CUDA(launch_gather(hi, u_out, HZ_F64, st));
  HZ_CUDA(cudaEventRecord(e1.e, st));
  HZ_CUDA(cudaStreamSynchronize(st));
  if (info) {
    hz_mixed_info inf{};
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0.e, e1.e);
    inf.cycles_done = cycles; inf.sweeps_lo = nlo; inf.sweeps_hi = nhi; inf.rel_residual = rel; inf.total_ms = ms;
    inf.dof_timesteps = (double)hi->L * hi->lay.lnx * hi->lay.lny * (double)opts->n_wh * (hi->n_t - 1) * (double)(nlo + nhi);
    *info = inf;
  }
  return HZ_OK;
}

extern "C" hz_status hz_minres_cycle(hz_ctx *ctx, const hz_minres_opts *opts, int *iters_out, double *res_out,
                                     hz_minres_info *info, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!opts) return fail(ctx, HZ_EINVAL, "hz_minres_cycle: NULL opts");
  if (!ctx->part) return fail(ctx, HZ_ESTATE, "hz_minres_cycle: call hz_partition first");
  const bool tile_ok = ctx->lay.variant == 1 && ctx->cl == 1 && ctx->mx == ctx->my && ctx->lay.TX * ctx->lay.TY <= 16 &&
                       ctx->lay.ntx * ctx->lay.nty <= 256 && !(ctx->p == 1 && ctx->mx == 1);
  if (ctx->lay.variant != 0 && !tile_ok)
    return fail(ctx, HZ_EUNSUPPORTED, "hz_minres_cycle: needs the one-DOF-per-thread partition or a register-blocked one with "
                                      "square tiles of at most 16 DOFs and at most 256 tiles per subdomain");
  if (!(opts->tol >= 0.0) || opts->max_iters < 0 || opts->relax < 0.0 || opts->relax > 1.0)
    return fail(ctx, HZ_EINVAL, "hz_minres_cycle: need tol >= 0, max_iters >= 0, relax in [0,1]");
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->prec == HZ_F32 ? minres_impl<float>(ctx, opts, iters_out, res_out, info, st)
                             : minres_impl<double>(ctx, opts, iters_out, res_out, info, st);
}

extern "C" hz_status hz_ddm_solve_gmres(hz_ctx *ctx, const hz_gmres_opts *opts, void *u_out, hz_gmres_info *info,
                                        void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!opts) return fail(ctx, HZ_EINVAL, "hz_ddm_solve_gmres: NULL opts");
  if (!ctx->part) return fail(ctx, HZ_ESTATE, "hz_ddm_solve_gmres: call hz_partition first");
  if (opts->n_wh < 1 || !(opts->relax > 0.0) || opts->relax > 1.0 || opts->restart < 1 || opts->restart > 1000 ||
      opts->max_steps < 0 || (opts->lin_history && opts->history_len < 0) || opts->n_polish < 0)
    return fail(ctx, HZ_EINVAL, "hz_ddm_solve_gmres: need n_wh >= 1, relax in (0,1], 1 <= restart <= 1000, max_steps >= 0, n_polish >= 0");
  cudaStream_t st = (cudaStream_t)stream;
  return ctx->prec == HZ_F32 ? gmres_impl<float>(ctx, opts, u_out, info, st) : gmres_impl<double>(ctx, opts, u_out, info, st);
}

extern "C" {

hz_status hz_residual(hz_ctx *ctx, const void *u_dev, hz_prec u_prec, double *rel_residual, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!u_dev || !rel_residual) return fail(ctx, HZ_EINVAL, "hz_residual: NULL u_dev or rel_residual");
  if (u_prec != HZ_F32 && u_prec != HZ_F64) return fail(ctx, HZ_EINVAL, "hz_residual: bad precision");
  double rel = 0.0;
  // the residual needs sx..E only through Geo fields that the kernel does not read when unpartitioned
  hz_status st = residual_impl(ctx, u_dev, u_prec, &rel, (cudaStream_t)stream);
  if (st != HZ_OK) return st;
  *rel_residual = rel;
  return HZ_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// hz_residual_static: hz_residual without any allocation (include/hz.h).  The block partial sums of k_helm /
// k_residual_quad and the reduced pair live in a file-scope device array instead of the context's lazily
// cudaMalloc'ed buffers.  In HOST code `g_res_static` is only the symbol's host-side stand-in, not a device address:
// the address the kernels get is resolved once per device with cudaGetSymbolAddress (that device current).
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_res_static[2 * (size_t)HZ_RESIDUAL_STATIC_MAX_BLOCKS + 32];
constexpr int kStaticMaxDevices = 64;
static double *g_res_static_ptr[kStaticMaxDevices] = {};
static std::mutex g_res_static_mu;

// device address of g_res_static on the CURRENT device (resolved on first use, then cached)
static cudaError_t res_static_address(double **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_res_static_mu);
  if (!g_res_static_ptr[dev]) {
    void *q = nullptr;
    e = cudaGetSymbolAddress(&q, g_res_static);
    if (e != cudaSuccess) return e;
    if (!q) return cudaErrorInvalidSymbol;
    g_res_static_ptr[dev] = static_cast<double *>(q);
  }
  *out = g_res_static_ptr[dev];
  return cudaSuccess;
}

// rel = sqrt(|r|^2 / |b|^2) (|b| = 0: sqrt(|r|^2)), the last step of residual_impl, on the device
static __global__ void k_rel_from_sums(const double *__restrict__ red, double *__restrict__ out) {
  if (threadIdx.x == 0 && blockIdx.x == 0) out[0] = red[1] > 0.0 ? sqrt(red[0] / red[1]) : sqrt(red[0]);
}

extern "C" {

int hz_residual_static_max_blocks(void) { return HZ_RESIDUAL_STATIC_MAX_BLOCKS; }

hz_status hz_residual_static_setup(hz_ctx *ctx) {
  if (!ctx) return HZ_EINVAL;
  double *scratch = nullptr;
  HZ_CUDA(res_static_address(&scratch));
  return HZ_OK;
}

hz_status hz_residual_static(hz_ctx *ctx, const void *u_dev, hz_prec u_prec, double *rel_residual_dev, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!u_dev || !rel_residual_dev) return fail(ctx, HZ_EINVAL, "hz_residual_static: NULL u_dev or rel_residual_dev");
  if (u_prec != HZ_F32 && u_prec != HZ_F64) return fail(ctx, HZ_EINVAL, "hz_residual_static: bad precision");
  cudaStream_t st = (cudaStream_t)stream;
  const long long total = (long long)ctx->npx * ctx->npy;
  const int bs = 256;
  const long long nb = ctx->general ? (total + bs - 1) / bs
                                    : (long long)((ctx->nx + 1 + kHelmBX - 1) / kHelmBX) * ((ctx->ny + 1 + kHelmBY - 1) / kHelmBY);
  if (nb > HZ_RESIDUAL_STATIC_MAX_BLOCKS) {
    char msg[192];
    std::snprintf(msg, sizeof(msg), "hz_residual_static: the mesh needs %lld partial-sum blocks, the static scratch holds %d "
                  "(HZ_RESIDUAL_STATIC_MAX_BLOCKS); use hz_residual", nb, HZ_RESIDUAL_STATIC_MAX_BLOCKS);
    return fail(ctx, HZ_EINVAL, msg);
  }
  double *part = nullptr;
  HZ_CUDA(res_static_address(&part));
  double *red = part + 2 * (size_t)HZ_RESIDUAL_STATIC_MAX_BLOCKS;
  // the array keeps the previous call's contents: the slots this call reads start at zero
  HZ_CUDA(cudaMemsetAsync(part, 0, (size_t)2 * nb * sizeof(double), st));
  HZ_CUDA(cudaMemsetAsync(red, 0, 2 * sizeof(double), st));
  if (ctx->general) {
    Geo g = make_geo(ctx);
    if (u_prec == HZ_F32)
      k_residual_quad<float><<<(unsigned)nb, bs, 0, st>>>(g, ctx->refq, ctx->d_vx, ctx->d_vy, ctx->d_c, ctx->d_fre, ctx->d_fim,
                                                          ctx->d_bc, (const float *)u_dev, part);
    else
      k_residual_quad<double><<<(unsigned)nb, bs, 0, st>>>(g, ctx->refq, ctx->d_vx, ctx->d_vy, ctx->d_c, ctx->d_fre, ctx->d_fim,
                                                           ctx->d_bc, (const double *)u_dev, part);
    HZ_CUDA(cudaGetLastError());
  } else if (u_prec == HZ_F32) {
    HZ_CUDA((launch_helm<float, double, 0>(ctx, nullptr, u_dev, part, nullptr, st, false)));
  } else {
    HZ_CUDA((launch_helm<double, double, 0>(ctx, nullptr, u_dev, part, nullptr, st, false)));
  }
  k_reduce2<<<1, 1024, 0, st>>>(part, (int)nb, red);
  HZ_CUDA(cudaGetLastError());
  k_rel_from_sums<<<1, 32, 0, st>>>(red, rel_residual_dev);
  HZ_CUDA(cudaGetLastError());
  return HZ_OK;
}

hz_status hz_get_subdomain_state(hz_ctx *ctx, double *u_sub_dev, double *lambda_dev, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!ctx->part) return fail(ctx, HZ_ESTATE, "hz_get_subdomain_state: call hz_partition first");
  cudaStream_t st = (cudaStream_t)stream;
  const int bs = 256;
  if (u_sub_dev) {
    const long long n = (long long)ctx->L * 2 * ctx->lay.lnx * ctx->lay.lny;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (ctx->prec == HZ_F32) k_state_get<float><<<nb, bs, 0, st>>>(ctx->lay, ctx->L, (const float *)ctx->d_usub, u_sub_dev);
    else k_state_get<double><<<nb, bs, 0, st>>>(ctx->lay, ctx->L, (const double *)ctx->d_usub, u_sub_dev);
    HZ_CUDA(cudaGetLastError());
  }
  if (lambda_dev) {
    const long long n = (long long)ctx->L * 8 * ctx->E;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (ctx->prec == HZ_F32) k_convert<float, double><<<nb, bs, 0, st>>>(n, (const float *)ctx->d_lam, lambda_dev);
    else k_convert<double, double><<<nb, bs, 0, st>>>(n, (const double *)ctx->d_lam, lambda_dev);
    HZ_CUDA(cudaGetLastError());
  }
  HZ_CUDA(cudaStreamSynchronize(st));
  return HZ_OK;
}

hz_status hz_set_subdomain_state(hz_ctx *ctx, const double *u_sub_dev, const double *lambda_dev, void *stream) {
  if (!ctx) return HZ_EINVAL;
  if (!ctx->part) return fail(ctx, HZ_ESTATE, "hz_set_subdomain_state: call hz_partition first");
  cudaStream_t st = (cudaStream_t)stream;
  const int bs = 256;
  if (u_sub_dev) {
    const long long n = (long long)ctx->L * 2 * ctx->lay.lnx * ctx->lay.lny;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (ctx->prec == HZ_F32) k_state_set<float><<<nb, bs, 0, st>>>(ctx->lay, ctx->L, (float *)ctx->d_usub, u_sub_dev);
    else k_state_set<double><<<nb, bs, 0, st>>>(ctx->lay, ctx->L, (double *)ctx->d_usub, u_sub_dev);
    HZ_CUDA(cudaGetLastError());
  }
  if (lambda_dev) {
    const long long n = (long long)ctx->L * 8 * ctx->E;
    const unsigned nb = (unsigned)((n + bs - 1) / bs);
    if (ctx->prec == HZ_F32) k_convert<double, float><<<nb, bs, 0, st>>>(n, lambda_dev, (float *)ctx->d_lam);
    else k_convert<double, double><<<nb, bs, 0, st>>>(n, lambda_dev, (double *)ctx->d_lam);
    HZ_CUDA(cudaGetLastError());
  }
  HZ_CUDA(cudaStreamSynchronize(st));
  return HZ_OK;
}

const char *hz_last_error(const hz_ctx *ctx) { return ctx ? ctx->err.c_str() : g_setup_error.c_str(); }

void hz_destroy(hz_ctx *ctx) {
  if (!ctx) return;
  free_partition(ctx);
  if (ctx->cap_stream) cudaStreamDestroy(ctx->cap_stream);
  if (ctx->s_ring) cudaStreamDestroy(ctx->s_ring);
  if (ctx->ev_rfork) cudaEventDestroy(ctx->ev_rfork);
  if (ctx->ev_rjoin) cudaEventDestroy(ctx->ev_rjoin);
  if (ctx->s_in) cudaStreamDestroy(ctx->s_in);
  if (ctx->s_out) cudaStreamDestroy(ctx->s_out);
  for (int b = 0; b < 2; ++b) {
    if (ctx->d_fstage[b]) cudaFree(ctx->d_fstage[b]);
    if (ctx->d_ubuf[b]) cudaFree(ctx->d_ubuf[b]);
    for (cudaEvent_t e : {ctx->ev_up[b], ctx->ev_build[b], ctx->ev_gather[b], ctx->ev_down[b]})
      if (e) cudaEventDestroy(e);
  }
  if (ctx->d_opk2) cudaFree(ctx->d_opk2);
  if (ctx->d_opy) cudaFree(ctx->d_opy);
  double **ptrs[] = {&ctx->d_c, &ctx->d_fre, &ctx->d_fim, &ctx->d_bc, &ctx->d_vx, &ctx->d_vy};
  for (double **q : ptrs) { if (*q) cudaFree(*q); *q = nullptr; }
  delete ctx;
}

}  // extern "C"
