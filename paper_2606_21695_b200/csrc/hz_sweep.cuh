// hz_sweep.cuh — the DDM-cycle ("sweep") kernels: Algorithm 1 of the paper on every
// subdomain at once, one thread block per subdomain, WaveHoltz as the subdomain
// solver.  Inside a sweep: no global memory in the time loop, no reductions, no
// device-wide synchronisation.
//
// This file: k_sweep_dof, one DOF per thread (PAPER.md:191-207 re-designed).  p^nu lives in a ping-pong
// shared-memory plane; each thread applies its own row of the assembled 1-D operators (2(2P+1)
// shared loads, one shared store and ONE __syncthreads per time step; no atomics).  The plane is stored
// contiguously (node t at word t): a band row is zero where it would leave the subdomain, so such a read may
// return any finite value (the neighbouring line, or the zero margin of P rows + P words around the plane) and
// consecutive lanes read consecutive words in both directions: no halo, no bounds checks, no bank conflicts.  The register-blocked
// variants are in hz_sweep_tile.cuh (rectangular tiles, uniform code) and hz_sweep_ws.cuh (square tiles,
// warp-specialised), the streamed fallback in hz_sweep_stream.cuh.
// On the uniform rectangular elements of all configs the stiffness is  A = (hy/hx) Wy (x) Kx + (hx/hy) Ky (x) Wx
// (assembled 1-D stiffness K and GLL weights W), so with the lumped mass m_j = (hx hy/4) wx_I wy_J
//     beta_j (A p)_j = gamma_j [ (4/hx^2) (Kx p)_I / wx_I + (4/hy^2) (Ky p)_J / wy_J ],   gamma_j = beta_j m_j,
// which is what all kernels evaluate (the "assembled line stencil" formulation, 2(P+2) FMAs per DOF).
#pragma once
#include "hz_line.cuh"

namespace hz {

// ------------------------------------------------------------------------------------------------
// Variant 0: one DOF per thread
// ------------------------------------------------------------------------------------------------
template <typename real, int P>
__global__ void __launch_bounds__(1024, 1) k_sweep_dof(const SweepArgs<real> A) {
  constexpr int B = 2 * P + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Tab4<real> *tab = reinterpret_cast<Tab4<real> *>(smem_raw);
  const int lnx = A.lay.lnx, lny = A.lay.lny, N = lnx * lny, NS = A.lay.NS;
  const int W = lnx, MARG = P * (lnx + 1);
  const int PL = (N + 2 * MARG + 3) / 4 * 4;  // <= (lnx + 2P)(lny + 2P), the size the host reserves per plane
  real *pb0 = reinterpret_cast<real *>(tab + A.n_t);
  real *pb1 = pb0 + PL;
  const int t = threadIdx.x, NT = blockDim.x, l = blockIdx.x;
  const bool act = t < N;
  const int i = act ? t % lnx : 0, j = act ? t / lnx : 0;

  for (int q = t; q < 2 * PL; q += NT) pb0[q] = real(0);
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

  const int center = MARG + (act ? t : 0);
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

}  // namespace hz
