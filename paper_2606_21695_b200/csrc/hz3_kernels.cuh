// hz3_kernels.cuh — kernels of the 3-D hexahedral variant (include/hz3.h).
// Same formulation as the 2-D one-DOF-per-thread kernel (hz_sweep.cuh): on uniform elements with lumped mass
//   beta_j (A p)_j = gamma_j [ (4/hx^2)(Kx p)_I / wx_I + (4/hy^2)(Ky p)_J / wy_J + (4/hz^2)(Kz p)_K / wz_K ],
// gamma_j = beta_j m_j, each term a (2P+1)-wide row of the assembled 1-D operator of that direction.
#pragma once
#include "hz_aux.cuh"
#include "hz_line.cuh"

namespace hz {

struct Geo3 {
  int nx, ny, nz, p, npx, npy, npz;
  int sx, sy, sz, ex, ey, ez;
  int lnx, lny, lnz, NS;  // nodes per subdomain side; slots per subdomain (>= lnx*lny*lnz)
  int F, FB;              // face stride of the lambda arrays; of the bc_lambda blocks
  double hx, hy, hz, omega, theta, sigma;
};

template <typename real>
struct Sweep3Args {
  Geo3 g;
  int n_t, n_wh, warm;
  real sigma, omega, cos_h, sin_h, two_over_nt;
  const Tab4<real> *tab;
  const real *gamma, *alpha, *bbf_re, *bbf_im;  // [L][NS]; bbf_im may be NULL
  real *u_sub;                                  // [L][2][NS]
  const real *lam;                              // [L][6][2][F]
  real *gout;                                   // [L][6][2][F]
  const real *k2face, *bs;                      // [L][6][F]
  const real *bandx, *bandy, *bandz;            // [ln*][2P+1]
};

// face index of subdomain node (i,j,k) on face f (hz3.h order)
__host__ __device__ inline int face_node(const Geo3 &g, int f, int i, int j, int k) {
  return f < 2 ? k * g.lny + j : (f < 4 ? k * g.lnx + i : j * g.lnx + i);
}
__host__ __device__ inline bool on_face(const Geo3 &g, int f, int i, int j, int k) {
  switch (f) {
    case 0: return i == 0;
    case 1: return i == g.lnx - 1;
    case 2: return j == 0;
    case 3: return j == g.lny - 1;
    case 4: return k == 0;
    default: return k == g.lnz - 1;
  }
}
// neighbour subdomain across face f, or -1 on the outer boundary
__host__ __device__ inline int face_neighbour(const Geo3 &g, int l, int f) {
  const int ix = l % g.sx, iy = (l / g.sx) % g.sy, iz = l / (g.sx * g.sy);
  switch (f) {
    case 0: return ix > 0 ? l - 1 : -1;
    case 1: return ix < g.sx - 1 ? l + 1 : -1;
    case 2: return iy > 0 ? l - g.sx : -1;
    case 3: return iy < g.sy - 1 ? l + g.sx : -1;
    case 4: return iz > 0 ? l - g.sx * g.sy : -1;
    default: return iz < g.sz - 1 ? l + g.sx * g.sy : -1;
  }
}

// ---------------------------------------------------------------------------------------------
// A0 in 3-D: per-subdomain operator data, one thread per (subdomain, node).  wx/wy/wz: assembled reference GLL
// weights of a subdomain side.  fp64, rounded once.
// ---------------------------------------------------------------------------------------------
template <typename real>
__global__ void k3_build(Geo3 g, const double *__restrict__ c, const double *__restrict__ f_re,
                         const double *__restrict__ f_im, const double *__restrict__ bc, const double *__restrict__ wx,
                         const double *__restrict__ wy, const double *__restrict__ wz, real *gamma, real *alpha,
                         real *bbf_re, real *bbf_im, real *k2face, real *bs) {
  const int N = g.lnx * g.lny * g.lnz;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)g.sx * g.sy * g.sz * N) return;
  const int l = (int)(gid / N), q = (int)(gid - (long long)l * N);
  const int i = q % g.lnx, j = (q / g.lnx) % g.lny, k = q / (g.lnx * g.lny);
  const int ix = l % g.sx, iy = (l / g.sx) % g.sy, iz = l / (g.sx * g.sy);
  const int I = ix * g.ex * g.p + i, J = iy * g.ey * g.p + j, K = iz * g.ez * g.p + k;
  const size_t gn = ((size_t)K * g.npy + J) * g.npx + I;
  const double cj = c[gn];
  const double m = 0.125 * g.hx * g.hy * g.hz * wx[i] * wy[j] * wz[k];
  const double M = m / (cj * cj);
  // face weights of this node: (h h / 4) x the two in-face reference weights
  double s[6];
  s[0] = s[1] = 0.25 * g.hy * g.hz * wy[j] * wz[k];
  s[2] = s[3] = 0.25 * g.hx * g.hz * wx[i] * wz[k];
  s[4] = s[5] = 0.25 * g.hx * g.hy * wx[i] * wy[j];
  double H = 0.0, bre = f_re[gn] * m, bim = f_im ? f_im[gn] * m : 0.0;
  for (int f = 0; f < 6; ++f) {
    if (!on_face(g, f, i, j, k)) continue;
    H += s[f] / cj;  // impedance on ALL faces of the subdomain
    if (bc && face_neighbour(g, l, f) < 0) {
      const int gi = f < 2 ? K * g.npy + J : (f < 4 ? K * g.npx + I : J * g.npx + I);
      bre += s[f] * bc[(size_t)(f * 2 + 0) * g.FB + gi];
      bim += s[f] * bc[(size_t)(f * 2 + 1) * g.FB + gi];
    }
  }
  const double den = M + g.theta * H, beta = g.sigma / den;
  const size_t o = (size_t)l * g.NS + q;
  gamma[o] = (real)(beta * m);
  alpha[o] = (real)((M - g.theta * H) / den);
  bbf_re[o] = (real)(beta * bre);
  if (bbf_im) bbf_im[o] = (real)(beta * bim);
  for (int f = 0; f < 6; ++f)
    if (on_face(g, f, i, j, k)) {
      const size_t e = ((size_t)l * 6 + f) * g.F + face_node(g, f, i, j, k);
      k2face[e] = (real)(2.0 * g.omega / cj);
      bs[e] = (real)(beta * s[f]);
    }
}

// ---------------------------------------------------------------------------------------------
// The sweep: Algorithm 1 on every subdomain, one thread block per subdomain, one thread per
// node.  p lives in two shared-memory volumes (ping-pong); pdot, v_r, v_i, the coefficients and the node's three
// band rows stay in registers; one barrier per step.  The volume is stored CONTIGUOUSLY (node t at word t, no halo
// inside): a band row has zeros where it would leave the subdomain, so what such a read returns (a finite value of
// another line, or the zero margin of P planes + P rows + P words before and after the volume) does not matter, and
// consecutive lanes read consecutive words in all three directions — no bank conflicts.
// ---------------------------------------------------------------------------------------------
template <typename real, int P, int MAXT>
__global__ void __launch_bounds__(MAXT) k3_sweep_dof(const Sweep3Args<real> A, const __grid_constant__ TabC<real> TC) {
  constexpr int B = 2 * P + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  real *vol = reinterpret_cast<real *>(smem_raw);
  const Geo3 &g = A.g;
  const int t = threadIdx.x, l = blockIdx.x;
  const int N = g.lnx * g.lny * g.lnz;
  const int SX = g.lnx, SXY = g.lnx * g.lny, MARG = P * (SXY + SX + 1);
  const int VOL = (N + 2 * MARG + 3) / 4 * 4;
  for (int q = t; q < 2 * VOL; q += blockDim.x) vol[q] = real(0);
  const bool act = t < N;
  const int i = act ? t % g.lnx : 0, j = act ? (t / g.lnx) % g.lny : 0, k = act ? t / (g.lnx * g.lny) : 0;
  const int pos = MARG + (act ? t : 0);
  real bx[B], by[B], bz[B];
#pragma unroll
  for (int d = 0; d < B; ++d) {
    bx[d] = act ? A.bandx[i * B + d] : real(0);
    by[d] = act ? A.bandy[j * B + d] : real(0);
    bz[d] = act ? A.bandz[k * B + d] : real(0);
  }
  const size_t o = (size_t)l * g.NS + t;
  real gam = real(0), alp = real(0), br = real(0), bi = real(0), ur = real(0), ui = real(0);
  if (act) {
    gam = A.gamma[o]; alp = A.alpha[o]; br = A.bbf_re[o];
    bi = A.bbf_im ? A.bbf_im[o] : real(0);
    // b from lambda^n on the interface faces; edge / corner nodes sum their faces (R13)
    for (int f = 0; f < 6; ++f)
      if (on_face(g, f, i, j, k) && face_neighbour(g, l, f) >= 0) {
        const int e = face_node(g, f, i, j, k);
        const real s = A.bs[((size_t)l * 6 + f) * g.F + e];
        br = fmaT(s, A.lam[((size_t)(l * 6 + f) * 2 + 0) * g.F + e], br);
        bi = fmaT(s, A.lam[((size_t)(l * 6 + f) * 2 + 1) * g.F + e], bi);
      }
    if (A.warm) {
      ur = A.u_sub[(size_t)l * 2 * g.NS + t];
      ui = A.u_sub[(size_t)l * 2 * g.NS + g.NS + t];
    }
  }
  __syncthreads();
  int cur = 0;
  for (int m = 0; m < A.n_wh; ++m) {
    const Tab4<real> t0 = A.n_t <= kTabCMax ? TC.t[0] : A.tab[0];
    real p = ur, pd = A.omega * (ui * A.cos_h - ur * A.sin_h);  // PAPER.md:168-170; readings R2, R8
    real vr = t0.k * p, vi = t0.kh * pd;
#pragma unroll 1
    for (int nu = 1; nu < A.n_t; ++nu) {
      const Tab4<real> tn = A.n_t <= kTabCMax ? TC.t[nu] : A.tab[nu];
      p = fmaT(A.sigma, pd, p);
      real *buf = vol + cur;
      if (act) buf[pos] = p;
      __syncthreads();
      real S = real(0);
#pragma unroll
      for (int d = 0; d < B; ++d) {
        S = fmaT(bx[d], buf[pos + (d - P)], S);
        S = fmaT(by[d], buf[pos + (d - P) * SX], S);
        S = fmaT(bz[d], buf[pos + (d - P) * SXY], S);
      }
      const real x = fmaT(bi, tn.s, fmaT(-gam, S, br * tn.c));
      pd = fmaT(alp, pd, x);
      vr = fmaT(tn.k, p, vr);
      vi = fmaT(tn.kh, pd, vi);
      cur = VOL - cur;
    }
    ur = A.two_over_nt * vr;  // eq. (7) prefactor (reading R4)
    ui = A.two_over_nt * vi;
  }
  if (!act) return;
  A.u_sub[(size_t)l * 2 * g.NS + t] = ur;
  A.u_sub[(size_t)l * 2 * g.NS + g.NS + t] = ui;
  // g = -lambda^n - 2 i k u on the interface faces (eq. (2), sign per reading R3)
  for (int f = 0; f < 6; ++f)
    if (on_face(g, f, i, j, k) && face_neighbour(g, l, f) >= 0) {
      const int e = face_node(g, f, i, j, k);
      const real k2 = A.k2face[((size_t)l * 6 + f) * g.F + e];
      const size_t a = ((size_t)(l * 6 + f) * 2) * g.F + e;
      A.gout[a] = fmaT(k2, ui, -A.lam[a]);
      A.gout[a + g.F] = fmaT(-k2, ur, -A.lam[a + g.F]);
    }
}

// ---------------------------------------------------------------------------------------------
// Column variant: one thread per (i,j) node COLUMN, its LNZ nodes along z in registers (state and coefficients).
// The z part of the operator is then register-only, with the band coefficients of the z direction as compile-time
// offsets into a by-value kernel parameter (constant bank operands); x and y parts read the shared volume as in
// k3_sweep_dof.  One third fewer shared loads per DOF and LNZ times fewer threads per barrier.
// ---------------------------------------------------------------------------------------------
constexpr int kColMaxZ = 10;
template <typename real>
struct BandZ {
  real z[kColMaxZ][2 * kMaxP + 1];  // z[k][d] = band row of z-node k (zero outside the subdomain)
};

template <typename real, int P, int LNZ, int MAXT>
__global__ void __launch_bounds__(MAXT) k3_sweep_col(const Sweep3Args<real> A, const __grid_constant__ BandZ<real> BZ,
                                                     const __grid_constant__ TabC<real> TC) {
  constexpr int B = 2 * P + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  real *vol = reinterpret_cast<real *>(smem_raw);
  const Geo3 &g = A.g;
  const int t = threadIdx.x, l = blockIdx.x;
  const int SX = g.lnx, SXY = g.lnx * g.lny, N = SXY * LNZ, MARG = P * (SXY + SX + 1);
  const int VOL = (N + 2 * MARG + 3) / 4 * 4;
  for (int q = t; q < 2 * VOL; q += blockDim.x) vol[q] = real(0);
  const bool act = t < SXY;
  const int i = act ? t % g.lnx : 0, j = act ? t / g.lnx : 0;
  const int pos = MARG + (act ? t : 0);
  real bx[B], by[B];
#pragma unroll
  for (int d = 0; d < B; ++d) {
    bx[d] = act ? A.bandx[i * B + d] : real(0);
    by[d] = act ? A.bandy[j * B + d] : real(0);
  }
  real gam[LNZ], alp[LNZ], br[LNZ], bi[LNZ], ur[LNZ], ui[LNZ];
#pragma unroll
  for (int k = 0; k < LNZ; ++k) {
    gam[k] = alp[k] = br[k] = bi[k] = ur[k] = ui[k] = real(0);
    if (act) {
      const size_t o = (size_t)l * g.NS + (size_t)k * SXY + t;
      gam[k] = A.gamma[o]; alp[k] = A.alpha[o]; br[k] = A.bbf_re[o];
      bi[k] = A.bbf_im ? A.bbf_im[o] : real(0);
      for (int f = 0; f < 6; ++f)  // b from lambda^n on the interface faces (R13)
        if (on_face(g, f, i, j, k) && face_neighbour(g, l, f) >= 0) {
          const int e = face_node(g, f, i, j, k);
          const real s = A.bs[((size_t)l * 6 + f) * g.F + e];
          br[k] = fmaT(s, A.lam[((size_t)(l * 6 + f) * 2 + 0) * g.F + e], br[k]);
          bi[k] = fmaT(s, A.lam[((size_t)(l * 6 + f) * 2 + 1) * g.F + e], bi[k]);
        }
      if (A.warm) {
        ur[k] = A.u_sub[(size_t)l * 2 * g.NS + (size_t)k * SXY + t];
        ui[k] = A.u_sub[(size_t)l * 2 * g.NS + g.NS + (size_t)k * SXY + t];
      }
    }
  }
  __syncthreads();
  int cur = 0;
  real p[LNZ], pd[LNZ], vr[LNZ], vi[LNZ];
  for (int m = 0; m < A.n_wh; ++m) {
    const Tab4<real> t0 = A.n_t <= kTabCMax ? TC.t[0] : A.tab[0];
#pragma unroll
    for (int k = 0; k < LNZ; ++k) {  // PAPER.md:168-170; readings R2, R8
      p[k] = ur[k];
      pd[k] = A.omega * (ui[k] * A.cos_h - ur[k] * A.sin_h);
      vr[k] = t0.k * p[k];
      vi[k] = t0.kh * pd[k];
    }
#pragma unroll 1
    for (int nu = 1; nu < A.n_t; ++nu) {
      const Tab4<real> tn = A.n_t <= kTabCMax ? TC.t[nu] : A.tab[nu];
      real *buf = vol + cur + pos;
#pragma unroll
      for (int k = 0; k < LNZ; ++k) {
        p[k] = fmaT(A.sigma, pd[k], p[k]);
        if (act) buf[k * SXY] = p[k];
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < LNZ; ++k) {
        const real *c = buf + k * SXY;
        real Sx = real(0), Sy = real(0), Sz = real(0);
#pragma unroll
        for (int d = 0; d < B; ++d) {
          Sx = fmaT(bx[d], c[d - P], Sx);
          Sy = fmaT(by[d], c[(d - P) * SX], Sy);
          if (k + d - P >= 0 && k + d - P < LNZ) Sz = fmaT(BZ.z[k][d], p[k + d - P < 0 ? 0 : (k + d - P >= LNZ ? 0 : k + d - P)], Sz);
        }
        const real S = (Sx + Sy) + Sz;
        const real x = fmaT(bi[k], tn.s, fmaT(-gam[k], S, br[k] * tn.c));
        pd[k] = fmaT(alp[k], pd[k], x);
        vr[k] = fmaT(tn.k, p[k], vr[k]);
        vi[k] = fmaT(tn.kh, pd[k], vi[k]);
      }
      cur = VOL - cur;
    }
#pragma unroll
    for (int k = 0; k < LNZ; ++k) {  // eq. (7) prefactor (reading R4)
      ur[k] = A.two_over_nt * vr[k];
      ui[k] = A.two_over_nt * vi[k];
    }
  }
  if (!act) return;
#pragma unroll
  for (int k = 0; k < LNZ; ++k) {
    A.u_sub[(size_t)l * 2 * g.NS + (size_t)k * SXY + t] = ur[k];
    A.u_sub[(size_t)l * 2 * g.NS + g.NS + (size_t)k * SXY + t] = ui[k];
    for (int f = 0; f < 6; ++f)  // g = -lambda^n - 2 i k u (eq. (2), sign per reading R3)
      if (on_face(g, f, i, j, k) && face_neighbour(g, l, f) >= 0) {
        const int e = face_node(g, f, i, j, k);
        const real k2 = A.k2face[((size_t)l * 6 + f) * g.F + e];
        const size_t a = ((size_t)(l * 6 + f) * 2) * g.F + e;
        A.gout[a] = fmaT(k2, ui[k], -A.lam[a]);
        A.gout[a + g.F] = fmaT(-k2, ur[k], -A.lam[a + g.F]);
      }
  }
}

// A8 in 3-D: lambda^{n+1}_{r,o} = (1-rho) lambda^n_{r,o} + rho g_{nb(r,o), opp(o)}; one thread per lambda entry.
template <typename real>
__global__ void k3_exchange(Geo3 g, real rho, real *__restrict__ lam, const real *__restrict__ gg) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)g.sx * g.sy * g.sz * 12 * g.F) return;
  const int e = (int)(gid % g.F), c = (int)((gid / g.F) % 2), o = (int)((gid / (2 * g.F)) % 6);
  const int r = (int)(gid / (12 * (long long)g.F));
  const int nb = face_neighbour(g, r, o);
  if (nb < 0) return;
  const real gv = gg[(((size_t)nb * 6 + (o ^ 1)) * 2 + c) * g.F + e];
  lam[gid] = (real(1) - rho) * lam[gid] + rho * gv;
}

// A7 / R19 in 3-D: mean of the copies at shared nodes, summed in (iz, iy, ix) order.
template <typename real, typename outT>
__global__ void k3_gather(Geo3 g, const real *__restrict__ u_sub, outT *__restrict__ u_out) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)g.npx * g.npy * g.npz;
  if (gid >= total) return;
  const int I = (int)(gid % g.npx), J = (int)((gid / g.npx) % g.npy), K = (int)(gid / ((long long)g.npx * g.npy));
  const int wx = g.ex * g.p, wy = g.ey * g.p, wz = g.ez * g.p;
  const int x1 = I / wx > g.sx - 1 ? g.sx - 1 : I / wx, y1 = J / wy > g.sy - 1 ? g.sy - 1 : J / wy;
  const int z1 = K / wz > g.sz - 1 ? g.sz - 1 : K / wz;
  const int x0 = (I == x1 * wx && x1 > 0) ? x1 - 1 : x1, y0 = (J == y1 * wy && y1 > 0) ? y1 - 1 : y1;
  const int z0 = (K == z1 * wz && z1 > 0) ? z1 - 1 : z1;
  double sr = 0.0, si = 0.0;
  int cnt = 0;
  for (int iz = z0; iz <= z1; ++iz)
    for (int iy = y0; iy <= y1; ++iy)
      for (int ix = x0; ix <= x1; ++ix) {
        const int l = (iz * g.sy + iy) * g.sx + ix;
        const int s = ((K - iz * wz) * g.lny + (J - iy * wy)) * g.lnx + (I - ix * wx);
        sr += (double)u_sub[(size_t)l * 2 * g.NS + s];
        si += (double)u_sub[(size_t)l * 2 * g.NS + g.NS + s];
        ++cnt;
      }
  u_out[gid] = (outT)(sr / cnt);
  u_out[total + gid] = (outT)(si / cnt);
}

// A10 in 3-D: residual of the unpartitioned system (4), fp64, one thread per global node; reduction as k_residual.
__device__ inline void line_sum(const Ref1D &ref, int P, int n_el, int X, const double *ur, const double *ui,
                                size_t base, size_t stride, double *kr, double *ki) {
  // sum over the elements containing node X of the row of K1 applied along the line (base + x*stride)
  const int a0 = X % P;
  const int e_hi = (X == n_el * P) ? n_el - 1 : X / P, e_lo = (a0 == 0 && X > 0) ? X / P - 1 : e_hi;
  double r = 0.0, im = 0.0;
  for (int e = e_lo; e <= e_hi; ++e) {
    const int a = X - e * P;
    for (int cc = 0; cc <= P; ++cc) {
      const size_t n = base + (size_t)(e * P + cc) * stride;
      r += ref.K[a][cc] * ur[n];
      im += ref.K[a][cc] * ui[n];
    }
  }
  *kr = r; *ki = im;
}
__device__ inline double asm_weight(const Ref1D &ref, int P, int n_el, int X) {
  const int a = X % P;
  if (a != 0) return ref.w[a];
  return (X > 0 && X < n_el * P) ? 2.0 * ref.w[0] : ref.w[0];
}

template <typename inT>
__global__ void k3_residual(Geo3 g, Ref1D ref, const double *__restrict__ c, const double *__restrict__ f_re,
                            const double *__restrict__ f_im, const double *__restrict__ bc,
                            const inT *__restrict__ u, double *__restrict__ ucopy, double *__restrict__ part) {
  // ucopy: the field in fp64 (filled by k3_to_f64 beforehand when inT is float); here u is read through it
  __shared__ double red[2][32];
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)g.npx * g.npy * g.npz;
  double r2 = 0.0, b2 = 0.0;
  if (gid < total) {
    const int I = (int)(gid % g.npx), J = (int)((gid / g.npx) % g.npy), K = (int)(gid / ((long long)g.npx * g.npy));
    const int P = g.p;
    const double *ur = ucopy, *ui = ucopy + total;
    const double wxI = asm_weight(ref, P, g.nx, I), wyJ = asm_weight(ref, P, g.ny, J), wzK = asm_weight(ref, P, g.nz, K);
    double kxr, kxi, kyr, kyi, kzr, kzi;
    line_sum(ref, P, g.nx, I, ur, ui, ((size_t)K * g.npy + J) * g.npx, 1, &kxr, &kxi);
    line_sum(ref, P, g.ny, J, ur, ui, (size_t)K * g.npy * g.npx + I, g.npx, &kyr, &kyi);
    line_sum(ref, P, g.nz, K, ur, ui, (size_t)J * g.npx + I, (size_t)g.npx * g.npy, &kzr, &kzi);
    const double ax = 0.5 * g.hy * g.hz / g.hx * wyJ * wzK, ay = 0.5 * g.hx * g.hz / g.hy * wxI * wzK;
    const double az = 0.5 * g.hx * g.hy / g.hz * wxI * wyJ;
    const double Aur = ax * kxr + ay * kyr + az * kzr, Aui = ax * kxi + ay * kyi + az * kzi;
    const double cj = c[gid];
    const double m = 0.125 * g.hx * g.hy * g.hz * wxI * wyJ * wzK, M = m / (cj * cj);
    const double s[3] = {0.25 * g.hy * g.hz * wyJ * wzK, 0.25 * g.hx * g.hz * wxI * wzK, 0.25 * g.hx * g.hy * wxI * wyJ};
    const bool onf[6] = {I == 0, I == g.npx - 1, J == 0, J == g.npy - 1, K == 0, K == g.npz - 1};
    double H = 0.0, bre = f_re[gid] * m, bim = f_im ? f_im[gid] * m : 0.0;
    for (int f = 0; f < 6; ++f)
      if (onf[f]) {
        H += s[f / 2] / cj;
        if (bc) {
          const int gi = f < 2 ? K * g.npy + J : (f < 4 ? K * g.npx + I : J * g.npx + I);
          bre += s[f / 2] * bc[(size_t)(f * 2 + 0) * g.FB + gi];
          bim += s[f / 2] * bc[(size_t)(f * 2 + 1) * g.FB + gi];
        }
      }
    const double u_r = ur[gid], u_i = ui[gid];
    const double w2M = g.omega * g.omega * M, wH = g.omega * H;
    const double rr = bre - Aur + (w2M * u_r - wH * u_i), ri = bim - Aui + (w2M * u_i + wH * u_r);
    r2 = rr * rr + ri * ri;
    b2 = bre * bre + bim * bim;
  }
  (void)u;
  for (int o = 16; o > 0; o >>= 1) {
    r2 += __shfl_down_sync(0xffffffffu, r2, o);
    b2 += __shfl_down_sync(0xffffffffu, b2, o);
  }
  const int w = threadIdx.x >> 5, ln = threadIdx.x & 31;
  if (ln == 0) { red[0][w] = r2; red[1][w] = b2; }
  __syncthreads();
  if (w == 0) {
    const int nw = blockDim.x >> 5;
    r2 = ln < nw ? red[0][ln] : 0.0;
    b2 = ln < nw ? red[1][ln] : 0.0;
    for (int o = 16; o > 0; o >>= 1) {
      r2 += __shfl_down_sync(0xffffffffu, r2, o);
      b2 += __shfl_down_sync(0xffffffffu, b2, o);
    }
    if (ln == 0) { part[2 * (size_t)blockIdx.x] = r2; part[2 * (size_t)blockIdx.x + 1] = b2; }
  }
}

template <typename inT>
__global__ void k3_to_f64(const inT *__restrict__ in, double *__restrict__ out, long long n) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid < n) out[gid] = (double)in[gid];
}

// state export in fp64: u_sub [L][2][N], lam [L][6][2][F]
template <typename real>
__global__ void k3_state_get(Geo3 g, const real *__restrict__ u_sub, const real *__restrict__ lam, double *u_out,
                             double *lam_out) {
  const int N = g.lnx * g.lny * g.lnz;
  const long long L = (long long)g.sx * g.sy * g.sz;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (u_out && gid < L * 2 * N) {
    const int q = (int)(gid % N), cpt = (int)((gid / N) % 2);
    const long long l = gid / (2 * N);
    u_out[gid] = (double)u_sub[(size_t)l * 2 * g.NS + (size_t)cpt * g.NS + q];
  }
  if (lam_out && gid < L * 12 * g.F) lam_out[gid] = (double)lam[gid];
}

}  // namespace hz
