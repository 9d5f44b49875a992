// hz_sweep.cuh — the DDM-cycle ("sweep") kernels: Algorithm 1 of the paper on every
// subdomain at once, one thread block per subdomain, WaveHoltz as the subdomain
// solver.  Inside a sweep: no global memory in the time loop, no reductions, no
// device-wide synchronisation.
//
// Two threading variants (re-designed for sm_100a):
//   k_sweep_dof   one DOF per thread.  p^nu lives in a ping-pong shared-memory plane with a halo; each
//                 thread applies its own row of the assembled 1-D operators (2(2P+1) shared loads, one
//                 shared store and ONE __syncthreads per time step; no atomics).
//   k_sweep_tile  k = (MX*P)*(MY*P) DOFs per thread, all state in registers.  A thread owns the MX x MY
//                 elements' "lower-left" nodes; per time step it publishes, per tile line, one raw value
//                 and one partial sum (the last element row restricted to its own nodes) and reads one of
//                 each from its 4 neighbours: 2(TX+TY) shared loads + 2(TX+TY) stores per k DOFs, one
//                 barrier per step.
// On the uniform rectangular elements of all configs the stiffness is  A = (hy/hx) Wy (x) Kx + (hx/hy) Ky (x) Wx
// (assembled 1-D stiffness K and GLL weights W), so with the lumped mass m_j = (hx hy/4) wx_I wy_J
//     beta_j (A p)_j = gamma_j [ (4/hx^2) (Kx p)_I / wx_I + (4/hy^2) (Ky p)_J / wy_J ],   gamma_j = beta_j m_j,
// which is what both kernels evaluate (the "assembled line stencil" formulation, 2(P+2) FMAs per DOF).
#pragma once
#include "hz_internal.h"

namespace hz {

template <typename real>
__device__ __forceinline__ real fmaT(real a, real b, real c);
template <>
__device__ __forceinline__ float fmaT<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <>
__device__ __forceinline__ double fmaT<double>(double a, double b, double c) { return fma(a, b, c); }

// ------------------------------------------------------------------------------------------------
// Variant 0: one DOF per thread
// ------------------------------------------------------------------------------------------------
template <typename real, int P>
__global__ void __launch_bounds__(1024, 1) k_sweep_dof(const SweepArgs<real> A) {
  constexpr int B = 2 * P + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Tab4<real> *tab = reinterpret_cast<Tab4<real> *>(smem_raw);
  const int lnx = A.lay.lnx, lny = A.lay.lny, N = lnx * lny, NS = A.lay.NS;
  const int W = lnx + 2 * P, H = lny + 2 * P;
  real *pb0 = reinterpret_cast<real *>(tab + A.n_t);
  real *pb1 = pb0 + W * H;
  const int t = threadIdx.x, NT = blockDim.x, l = blockIdx.x;
  const bool act = t < N;
  const int i = act ? t % lnx : 0, j = act ? t / lnx : 0;

  for (int q = t; q < 2 * W * H; q += NT) pb0[q] = real(0);
  for (int q = t; q < A.n_t; q += NT) tab[q] = A.tab[q];

  real cx[B], cy[B];
#pragma unroll
  for (int d = 0; d < B; ++d) {
    cx[d] = act ? A.bandx[i * B + d] : real(0);
    cy[d] = act ? A.bandy[j * B + d] : real(0);
  }
  const size_t base = (size_t)l * NS + t;
  real gam = 0, al = 0, bbr = 0, bbi = 0, ur = 0, ui = 0;
  // interface data of this thread's node: up to two sides (corner)
  const int six = l % A.sx, siy = l / A.sx;
  const bool nbW = six > 0, nbE = six < A.sx - 1, nbS = siy > 0, nbN = siy < A.sy - 1;
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;
  const bool onW = act && i == 0 && nbW, onE = act && i == lnx - 1 && nbE;
  const bool onS = act && j == 0 && nbS, onN = act && j == lny - 1 && nbN;
  real lW_r = 0, lW_i = 0, lE_r = 0, lE_i = 0, lS_r = 0, lS_i = 0, lN_r = 0, lN_i = 0;
  if (act) {
    gam = A.gamma[base];
    al = A.alpha[base];
    bbr = A.bbf_re[base];
    if (A.bbf_im) bbi = A.bbf_im[base];
    if (A.warm) {
      ur = A.u_sub[(size_t)l * 2 * NS + t];
      ui = A.u_sub[(size_t)l * 2 * NS + NS + t];
    }
    // Assemble b from f and lambda^n: b_j = f_j m_j + sum_sides s_j lambda_j, times beta_j
    if (onW) { lW_r = A.lam[lbase + (kSideW * 2 + 0) * A.E + j]; lW_i = A.lam[lbase + (kSideW * 2 + 1) * A.E + j];
               real s = A.bs[ebase + kSideW * A.E + j]; bbr = fmaT(s, lW_r, bbr); bbi = fmaT(s, lW_i, bbi); }
    if (onE) { lE_r = A.lam[lbase + (kSideE * 2 + 0) * A.E + j]; lE_i = A.lam[lbase + (kSideE * 2 + 1) * A.E + j];
               real s = A.bs[ebase + kSideE * A.E + j]; bbr = fmaT(s, lE_r, bbr); bbi = fmaT(s, lE_i, bbi); }
    if (onS) { lS_r = A.lam[lbase + (kSideS * 2 + 0) * A.E + i]; lS_i = A.lam[lbase + (kSideS * 2 + 1) * A.E + i];
               real s = A.bs[ebase + kSideS * A.E + i]; bbr = fmaT(s, lS_r, bbr); bbi = fmaT(s, lS_i, bbi); }
    if (onN) { lN_r = A.lam[lbase + (kSideN * 2 + 0) * A.E + i]; lN_i = A.lam[lbase + (kSideN * 2 + 1) * A.E + i];
               real s = A.bs[ebase + kSideN * A.E + i]; bbr = fmaT(s, lN_r, bbr); bbi = fmaT(s, lN_i, bbi); }
  }
  __syncthreads();

  const int center = (j + P) * W + (i + P);
  const real sigma = A.sigma;
  int par = 0;
  for (int m = 0; m < A.n_wh; ++m) {
    // WaveHoltz init (readings R2, R8)
    real p = ur;
    real pd = A.omega * (ui * A.cos_h - ur * A.sin_h);
    const Tab4<real> t0 = tab[0];
    real vr = t0.k * p;
    real vi = t0.kh * pd;
    for (int nu = 1; nu < A.n_t; ++nu) {
      p = fmaT(sigma, pd, p);
      real *buf = par ? pb1 : pb0;
      par ^= 1;
      if (act) buf[center] = p;
      __syncthreads();
      real S = real(0);  // (Lx p + Ly p)_j
#pragma unroll
      for (int d = 0; d < B; ++d) {
        S = fmaT(cx[d], buf[center + (d - P)], S);
        S = fmaT(cy[d], buf[center + (d - P) * W], S);
      }
      const Tab4<real> tn = tab[nu];
      // pdot <- alpha pdot + beta(-A p + Re{b e^{-2 pi i nu/N_t}})   (readings R5, R7)
      const real src = fmaT(bbr, tn.c, bbi * tn.s);
      pd = fmaT(al, pd, fmaT(-gam, S, src));
      vr = fmaT(tn.k, p, vr);   // PAPER.md:177 with the sign of eq. (7) (reading R2)
      vi = fmaT(tn.kh, pd, vi);
    }
    ur = A.two_over_nt * vr;  // eq. (7) prefactor (reading R4)
    ui = A.two_over_nt * vi;
  }
  if (act) {
    A.u_sub[(size_t)l * 2 * NS + t] = ur;
    A.u_sub[(size_t)l * 2 * NS + NS + t] = ui;
    // outgoing interface data g = -lambda^n - 2 i k u  (eq. (2); sign per reading R3)
    if (onW) { real k2 = A.k2edge[ebase + kSideW * A.E + j];
               A.gout[lbase + (kSideW * 2 + 0) * A.E + j] = fmaT(k2, ui, -lW_r);
               A.gout[lbase + (kSideW * 2 + 1) * A.E + j] = fmaT(-k2, ur, -lW_i); }
    if (onE) { real k2 = A.k2edge[ebase + kSideE * A.E + j];
               A.gout[lbase + (kSideE * 2 + 0) * A.E + j] = fmaT(k2, ui, -lE_r);
               A.gout[lbase + (kSideE * 2 + 1) * A.E + j] = fmaT(-k2, ur, -lE_i); }
    if (onS) { real k2 = A.k2edge[ebase + kSideS * A.E + i];
               A.gout[lbase + (kSideS * 2 + 0) * A.E + i] = fmaT(k2, ui, -lS_r);
               A.gout[lbase + (kSideS * 2 + 1) * A.E + i] = fmaT(-k2, ur, -lS_i); }
    if (onN) { real k2 = A.k2edge[ebase + kSideN * A.E + i];
               A.gout[lbase + (kSideN * 2 + 0) * A.E + i] = fmaT(k2, ui, -lN_r);
               A.gout[lbase + (kSideN * 2 + 1) * A.E + i] = fmaT(-k2, ur, -lN_i); }
  }
}

// ------------------------------------------------------------------------------------------------
// Variant 1: k = (MX*P)*(MY*P) DOFs per thread, register-blocked
// ------------------------------------------------------------------------------------------------
template <typename real, int P, int MX, int MY, bool CSM, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_sweep_tile(const SweepArgs<real> A) {
  constexpr int TX = MX * P, TY = MY * P, KT = TX * TY;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Tab4<real> *tab = reinterpret_cast<Tab4<real> *>(smem_raw);
  const int t = threadIdx.x, NT = blockDim.x, l = blockIdx.x;
  const int NS1 = NT + 1;  // exchange arrays carry one extra always-zero slot at index NT
  // per buffer: PX[TY], RX[TY], PY[TX], RY[TX], each NS1 long
  constexpr int NARR = 2 * TY + 2 * TX;
  real *xb0 = reinterpret_cast<real *>(tab + A.n_t);
  real *xb1 = xb0 + NARR * NS1;
  // CSM: the read-only per-DOF coefficients gamma_j and beta_j Re b_j live in shared memory (large
  // subdomains whose state alone fills the register file); otherwise they are registers.
  real *csm = xb1 + NARR * NS1;  // [2][KT][NT]
  const int ntx = A.lay.ntx, nty = A.lay.nty, NS = A.lay.NS;
  const int lnx = A.lay.lnx, lny = A.lay.lny;
  const bool act = t < ntx * nty;
  const int tx = act ? t % ntx : 0, ty = act ? t / ntx : 0;

  for (int q = t; q < 2 * NARR * NS1; q += NT) xb0[q] = real(0);
  for (int q = t; q < A.n_t; q += NT) tab[q] = A.tab[q];

  // neighbour slots (NT = the zero slot)
  const int iL = (act && tx > 0) ? t - 1 : NT;
  const int iR = (act && tx < ntx - 1) ? t + 1 : NT;
  const int iD = (act && ty > 0) ? t - ntx : NT;
  const int iU = (act && ty < nty - 1) ? t + ntx : NT;
  // first node of the tile: one-sided at the subdomain ends (assembled weight w_0 instead of 2 w_0)
  const bool hasL = tx > 0, hasR = tx < ntx - 1, hasD = ty > 0, hasU = ty < nty - 1;
  const real d0x = (hasR ? A.ex1.k0[0] : real(0)) + (hasL ? A.ex1.kp[P] : real(0));
  const real d0y = (hasU ? A.ey1.k0[0] : real(0)) + (hasD ? A.ey1.kp[P] : real(0));
  const real s0x = (hasL && hasR) ? real(1) : real(2);
  const real s0y = (hasD && hasU) ? real(1) : real(2);

  real p[TY][TX], pd[TY][TX], vr[TY][TX], vi[TY][TX];
  real gam[CSM ? 1 : TY][CSM ? 1 : TX], bbr[CSM ? 1 : TY][CSM ? 1 : TX];
  real ur[TY][TX], ui[TY][TX];
  // boundary-only data: column 0 (nodes (0,b)) and row 0 (nodes (a,0), a >= 1)
  real alc[TY], bic[TY], alr[TX], bir[TX];
  const size_t base = (size_t)l * NS + t;
#pragma unroll
  for (int b = 0; b < TY; ++b)
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      const size_t o = base + (size_t)(b * TX + a) * NT;
      if (CSM) {
        csm[(b * TX + a) * NT + t] = A.gamma[o];
        csm[(KT + b * TX + a) * NT + t] = A.bbf_re[o];
      } else {
        gam[b][a] = A.gamma[o];
        bbr[b][a] = A.bbf_re[o];
      }
      if (A.warm) {
        ur[b][a] = A.u_sub[(size_t)l * 2 * NS + (size_t)(b * TX + a) * NT + t];
        ui[b][a] = A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * TX + a) * NT + t];
      } else {
        ur[b][a] = real(0);
        ui[b][a] = real(0);
      }
    }
#pragma unroll
  for (int b = 0; b < TY; ++b) {
    const size_t o = base + (size_t)(b * TX) * NT;
    alc[b] = A.alpha[o];
    bic[b] = A.bbf_im ? A.bbf_im[o] : real(0);
  }
#pragma unroll
  for (int a = 0; a < TX; ++a) {
    const size_t o = base + (size_t)a * NT;
    alr[a] = A.alpha[o];
    bir[a] = A.bbf_im ? A.bbf_im[o] : real(0);
  }
  // Assemble b from lambda^n.  Boundary nodes are column 0 of the first/last tile column
  // and row 0 of the first/last tile row.
  const int six = l % A.sx, siy = l / A.sx;
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;
  int sideX = -1, sideY = -1;  // interface side carried by this tile's column 0 / row 0
  if (act && tx == 0 && six > 0) sideX = kSideW;
  if (act && tx == ntx - 1 && six < A.sx - 1) sideX = kSideE;
  if (act && ty == 0 && siy > 0) sideY = kSideS;
  if (act && ty == nty - 1 && siy < A.sy - 1) sideY = kSideN;
  real lcr[TY], lci[TY], lrr[TX], lri[TX];  // lambda^n on column 0 / row 0
#pragma unroll
  for (int b = 0; b < TY; ++b) { lcr[b] = 0; lci[b] = 0; }
#pragma unroll
  for (int a = 0; a < TX; ++a) { lrr[a] = 0; lri[a] = 0; }
  if (sideX >= 0) {
#pragma unroll
    for (int b = 0; b < TY; ++b) {
      const int j = ty * TY + b;
      if (j < lny) {
        lcr[b] = A.lam[lbase + (sideX * 2 + 0) * A.E + j];
        lci[b] = A.lam[lbase + (sideX * 2 + 1) * A.E + j];
        const real s = A.bs[ebase + sideX * A.E + j];
        if (CSM) csm[(KT + b * TX) * NT + t] = fmaT(s, lcr[b], csm[(KT + b * TX) * NT + t]);
        else bbr[b][0] = fmaT(s, lcr[b], bbr[b][0]);
        bic[b] = fmaT(s, lci[b], bic[b]);
      }
    }
  }
  if (sideY >= 0) {
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      const int i = tx * TX + a;
      if (i < lnx) {
        lrr[a] = A.lam[lbase + (sideY * 2 + 0) * A.E + i];
        lri[a] = A.lam[lbase + (sideY * 2 + 1) * A.E + i];
        const real s = A.bs[ebase + sideY * A.E + i];
        if (CSM) csm[(KT + a) * NT + t] = fmaT(s, lrr[a], csm[(KT + a) * NT + t]);
        else bbr[0][a] = fmaT(s, lrr[a], bbr[0][a]);
        if (a == 0) bic[0] = fmaT(s, lri[a], bic[0]);
        else bir[a] = fmaT(s, lri[a], bir[a]);
      }
    }
  }
  __syncthreads();

  const real sigma = A.sigma;
  int par = 0;
  for (int m = 0; m < A.n_wh; ++m) {
    const Tab4<real> t0 = tab[0];
#pragma unroll
    for (int b = 0; b < TY; ++b)
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        p[b][a] = ur[b][a];
        pd[b][a] = A.omega * (ui[b][a] * A.cos_h - ur[b][a] * A.sin_h);
        vr[b][a] = t0.k * p[b][a];
        vi[b][a] = t0.kh * pd[b][a];
      }
#pragma unroll 1
    for (int nu = 1; nu < A.n_t; ++nu) {
      real *xb = par ? xb1 : xb0;
      par ^= 1;
      real *PX = xb, *RX = xb + TY * NS1, *PY = xb + 2 * TY * NS1, *RY = xb + (2 * TY + TX) * NS1;
      // p <- p + sigma pdot, then publish what the neighbours need
#pragma unroll
      for (int b = 0; b < TY; ++b)
#pragma unroll
        for (int a = 0; a < TX; ++a) p[b][a] = fmaT(sigma, pd[b][a], p[b][a]);
#pragma unroll
      for (int b = 0; b < TY; ++b) {
        real s = A.ex1.kp[0] * p[b][(MX - 1) * P];
#pragma unroll
        for (int c = 1; c < P; ++c) s = fmaT(A.ex1.kp[c], p[b][(MX - 1) * P + c], s);
        PX[b * NS1 + t] = s;
        RX[b * NS1 + t] = p[b][0];
      }
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        real s = A.ey1.kp[0] * p[(MY - 1) * P][a];
#pragma unroll
        for (int c = 1; c < P; ++c) s = fmaT(A.ey1.kp[c], p[(MY - 1) * P + c][a], s);
        PY[a * NS1 + t] = s;
        RY[a * NS1 + t] = p[0][a];
      }
      __syncthreads();
      real S[TY][TX];
      // x direction: line b of the tile is q[0..TX-1] (own) + q[TX] (first column of the right neighbour)
#pragma unroll
      for (int b = 0; b < TY; ++b) {
        real q[TX + 1];
#pragma unroll
        for (int a = 0; a < TX; ++a) q[a] = p[b][a];
        q[TX] = RX[b * NS1 + iR];
        const real pin = PX[b * NS1 + iL];
        {  // first node of the tile
          real T = fmaT(d0x, q[0], pin);
#pragma unroll
          for (int c = 1; c <= P; ++c) T = fmaT(A.ex1.k0[c], q[c], T);
          S[b][0] = s0x * T;
        }
#pragma unroll
        for (int e = 0; e < MX; ++e) {
#pragma unroll
          for (int a = 1; a < P; ++a) {  // element-interior nodes
            real T = A.ex1.kin[a][0] * q[e * P];
#pragma unroll
            for (int c = 1; c <= P; ++c) T = fmaT(A.ex1.kin[a][c], q[e * P + c], T);
            S[b][e * P + a] = T;
          }
          if (e > 0) {  // node shared by elements e-1 and e of the tile
            real T = (A.ex1.k0[0] + A.ex1.kp[P]) * q[e * P];
#pragma unroll
            for (int c = 0; c < P; ++c) T = fmaT(A.ex1.kp[c], q[(e - 1) * P + c], T);
#pragma unroll
            for (int c = 1; c <= P; ++c) T = fmaT(A.ex1.k0[c], q[e * P + c], T);
            S[b][e * P] = T;
          }
        }
      }
      // y direction
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        real q[TY + 1];
#pragma unroll
        for (int b = 0; b < TY; ++b) q[b] = p[b][a];
        q[TY] = RY[a * NS1 + iU];
        const real pin = PY[a * NS1 + iD];
        {
          real T = fmaT(d0y, q[0], pin);
#pragma unroll
          for (int c = 1; c <= P; ++c) T = fmaT(A.ey1.k0[c], q[c], T);
          S[0][a] = fmaT(s0y, T, S[0][a]);
        }
#pragma unroll
        for (int e = 0; e < MY; ++e) {
#pragma unroll
          for (int b = 1; b < P; ++b) {
            real T = S[e * P + b][a];
#pragma unroll
            for (int c = 0; c <= P; ++c) T = fmaT(A.ey1.kin[b][c], q[e * P + c], T);
            S[e * P + b][a] = T;
          }
          if (e > 0) {
            real T = fmaT(A.ey1.k0[0] + A.ey1.kp[P], q[e * P], S[e * P][a]);
#pragma unroll
            for (int c = 0; c < P; ++c) T = fmaT(A.ey1.kp[c], q[(e - 1) * P + c], T);
#pragma unroll
            for (int c = 1; c <= P; ++c) T = fmaT(A.ey1.k0[c], q[e * P + c], T);
            S[e * P][a] = T;
          }
        }
      }
      const Tab4<real> tn = tab[nu];
      // pdot, filter
#pragma unroll
      for (int b = 0; b < TY; ++b)
#pragma unroll
        for (int a = 0; a < TX; ++a) {
          const real g_ = CSM ? csm[(b * TX + a) * NT + t] : gam[CSM ? 0 : b][CSM ? 0 : a];
          const real r_ = CSM ? csm[(KT + b * TX + a) * NT + t] : bbr[CSM ? 0 : b][CSM ? 0 : a];
          real x = fmaT(-g_, S[b][a], r_ * tn.c);
          if (a == 0) {
            x = fmaT(bic[b], tn.s, x);
            pd[b][a] = fmaT(alc[b], pd[b][a], x);
          } else if (b == 0) {
            x = fmaT(bir[a], tn.s, x);
            pd[b][a] = fmaT(alr[a], pd[b][a], x);
          } else {
            pd[b][a] += x;
          }
          vr[b][a] = fmaT(tn.k, p[b][a], vr[b][a]);
          vi[b][a] = fmaT(tn.kh, pd[b][a], vi[b][a]);
        }
    }
#pragma unroll
    for (int b = 0; b < TY; ++b)
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        ur[b][a] = A.two_over_nt * vr[b][a];
        ui[b][a] = A.two_over_nt * vi[b][a];
      }
  }
  // store u_l (A7) and the outgoing interface data (A6)
#pragma unroll
  for (int b = 0; b < TY; ++b)
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      A.u_sub[(size_t)l * 2 * NS + (size_t)(b * TX + a) * NT + t] = ur[b][a];
      A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * TX + a) * NT + t] = ui[b][a];
    }
  if (sideX >= 0) {
#pragma unroll
    for (int b = 0; b < TY; ++b) {
      const int j = ty * TY + b;
      if (j < lny) {
        const real k2 = A.k2edge[ebase + sideX * A.E + j];
        A.gout[lbase + (sideX * 2 + 0) * A.E + j] = fmaT(k2, ui[b][0], -lcr[b]);
        A.gout[lbase + (sideX * 2 + 1) * A.E + j] = fmaT(-k2, ur[b][0], -lci[b]);
      }
    }
  }
  if (sideY >= 0) {
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      const int i = tx * TX + a;
      if (i < lnx) {
        const real k2 = A.k2edge[ebase + sideY * A.E + i];
        A.gout[lbase + (sideY * 2 + 0) * A.E + i] = fmaT(k2, ui[0][a], -lrr[a]);
        A.gout[lbase + (sideY * 2 + 1) * A.E + i] = fmaT(-k2, ur[0][a], -lri[a]);
      }
    }
  }
}

}  // namespace hz
